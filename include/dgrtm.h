/* dgrtm.h - C ABI of libdgrtm: nodal discontinuous Galerkin time-domain (DGTD) acoustic solver and
 * reverse-time migration (RTM) on unstructured tetrahedra, hand-written CUDA for sm_100a (B200).
 *
 * Method: Modave, St-Cyr, Mulder, Warburton, arXiv 1506.00907 ("the paper"; PAPER.md = its text).
 * Every entry point cites the passage that defines the operation.  Readings of silent / garbled
 * passages are numbered Q1..Q16 in DESIGN.md.
 *
 * Conventions
 *  - plain C, opaque handle dg_ctx*.  Every call returns int: 0 = OK, negative = error code below;
 *    dg_last_error(ctx) returns a message owned by the ctx.  No exception or abort crosses the ABI.
 *  - HOST pointers everywhere except dg_bind_workspace / rtm_bind_history, which take DEVICE pointers
 *    (the caller owns device memory, e.g. a torch uint8 tensor) and a cudaStream_t passed as void*.
 *  - input arrays are borrowed for the duration of the call and copied; outputs go to caller-allocated
 *    buffers.  Indices are 0-based int32.  Coordinates, material and field values cross the ABI as
 *    double regardless of the compute precision (rounded once inside).
 *  - element order and node order of every array crossing the ABI is the USER's (the order of EToV
 *    and of dg_get_nodes); the internal level-sorted, 32-element-blocked layout never shows.
 *  - field layout q[k][field][n], field 0 = p, 1..3 = v_x, v_y, v_z (eqs (1)-(2)).
 *  - levels: 0 = coarsest (the paper's l = 1) .. L-1 = finest.
 *  - all kernels are enqueued on the bound stream; calls that return data synchronise that stream.
 *  - a ctx is not thread-safe; distinct ctxs are independent.
 */
#ifndef DGRTM_H
#define DGRTM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dg_ctx dg_ctx;

enum {
  DG_OK = 0,
  DG_ERR_ARG = -1,         /* NULL / out-of-range argument or size */
  DG_ERR_MESH = -2,        /* degenerate, negatively oriented or non-conforming mesh */
  DG_ERR_STATE = -3,       /* call out of order (e.g. dg_step before dg_set_model / bind) */
  DG_ERR_CUDA = -4,        /* CUDA runtime error (message in dg_last_error) */
  DG_ERR_NOMEM = -5,       /* bound workspace / history too small */
  DG_ERR_UNSUPPORTED = -6  /* N outside 1..6, precision not 32/64, ... */
};

/* boundary-condition types of a boundary face (eq (3); exterior states: reading Q6) */
enum { DG_BC_FREE = 1, DG_BC_ABSORBING = 2, DG_BC_RIGID = 3, DG_BC_PRESCRIBED = 4 };
enum { DG_INTEGRATOR_AB3 = 0, DG_INTEGRATOR_LSERK4 = 1 };
enum { DG_WAVELET_RICKER = 0 };
/* imaging condition (bit 0: characteristic variables (7) instead of p_S p_R (4)) and time quadrature (bit 1: the
 * trapezoid rule (21) PAPER.md:178-180 instead of the Adams-Bashforth-consistent integral (22)-(24)) */
enum { DG_IMAGING_CLASSICAL = 0, DG_IMAGING_CHARACTERISTIC = 1, DG_IMAGING_CLASSICAL_TRAPEZOID = 2,
       DG_IMAGING_CHARACTERISTIC_TRAPEZOID = 3 };
enum { DG_RHS_VOLUME = 0, DG_RHS_SURFACE = 1, DG_RHS_TOTAL = 2 };

const char* dg_version(void);
/* Message of the last failed call on this ctx (or of the last failed dg_mesh_create if ctx==NULL). */
const char* dg_last_error(const dg_ctx* ctx);

/* ---- setup -------------------------------------------------------------------------------------
 * dg_mesh_create: nodal DG space of order N (N_p=(N+1)(N+2)(N+3)/6 warp-and-blend nodes, eqs (9)-(10)
 * PAPER.md:84-96) on the K tetrahedra EToV[K][4] with vertices VX[Nv][3]; builds D_r,D_s,D_t, L_f
 * (App. A 593-612), geometric factors (App. A 606-624, reading Q3), face connectivity
 * and the boundary-face list (host, fp64).  precision = 32 or 64 selects the device arithmetic.
 * face_bc[K][4] (may be NULL) gives the type of each BOUNDARY face (0 -> default_bc); entries of
 * interior faces are ignored.  Tets with non-positive volume -> DG_ERR_MESH (never re-ordered). */
int dg_mesh_create(dg_ctx** out, int N, int precision, int64_t K, int64_t Nv, const int32_t* EToV,
                   const double* VX, const int8_t* face_bc, int default_bc);
void dg_destroy(dg_ctx* ctx);

/* dg_set_model: piecewise-constant rho[K], c[K] (replaces phyDB/phyMap PAPER.md:258).
 * dt_k = cfl*l_k/((N+1)^2 c_k), dt_local = min_k dt_k, multi-rate levels with at most
 * one level between face neighbours (reading Q9), level-sorted device layout.
 * nlevels = 1 -> single rate.  Must precede dg_workspace_bytes. */
int dg_set_model(dg_ctx* ctx, const double* rho, const double* c, int nlevels, double cfl);
/* AB3 / multi-rate AB3 (eqs (18)-(19) PAPER.md:156-166, Alg. 1; default) or the
 * five-stage LSERK4 (not in the paper; BASELINE.json config 1, reading Q8; single rate only). */
int dg_set_integrator(dg_ctx* ctx, int integrator);
/* Overrides dt_local (default: the CFL value of dg_set_model).  Testing aid (convergence in dt). */
int dg_set_dt(dg_ctx* ctx, double dt_local);

/* Point source f(t) delta(x-x0) L2-projected on the element containing x0 (eq (15) PAPER.md:122-128,
 * scaling of eq (1): reading Q5; owner element: reading Q11).  Ricker f(t) = amp (1-2a) exp(-a),
 * a = (pi f0 (t-tp))^2. */
int dg_set_source(dg_ctx* ctx, const double x0[3], int wavelet, double f0, double tp, double amp);
/* nr receivers xr[nr][3]: sampling rows l_n(x_r) and injection weights M_k^-1 l(x_r) (eq (15)).  The receiver-sized part
 * of the RTM region holds max(nr at bind time, rtm_set_receiver_capacity) receivers: a new receiver set within that
 * capacity keeps the region (image, q(t_f) and trace history untouched: the gathers of a survey stack in place,
 * PAPER.md:61, 460, 478); a larger one unbinds it (rtm_history_bytes / rtm_bind_history again; the image restarts). */
int dg_set_receivers(dg_ctx* ctx, int64_t nr, const double* xr);

/* Device memory.  The library allocates none: query, allocate (e.g. a torch tensor), bind.
 * dptr must be 256-byte aligned device memory of at least n bytes that stays valid until dg_destroy
 * or the next bind; stream is a cudaStream_t (NULL = legacy default stream).  Binding uploads all
 * tables and zeroes the fields (state = rest at t = 0). */
int dg_workspace_bytes(dg_ctx* ctx, size_t* n);
int dg_bind_workspace(dg_ctx* ctx, void* dptr, size_t n, void* cuda_stream);

/* ---- time stepping ------------------------------------------------------------------------------
 * dg_set_state: nodal fields q[K][4][Np] at time t0; right-hand-side history cleared (AB start-up by
 * AB1, AB2: reading Q7); exposed traces (p, n.v) refreshed. */
int dg_set_state(dg_ctx* ctx, const double* q, double t0);
/* Advance nsteps GLOBAL steps (= 2^(L-1) fine steps of dt_local each) forward in time with the point
 * source on (if set): per fine step the volume + surface right-hand side (eqs (13)-(14) PAPER.md:
 * 113-118, penalties (11)-(12) PAPER.md:100-111, Algs 2-3) of the levels that sit at the step start,
 * the update (18) of the levels that land on the step end and the half-step traces (19) of their
 * not-updated coarse neighbours (Alg. 1, Alg. 4).  Asynchronous on the stream. */
int dg_step(dg_ctx* ctx, int nsteps);
/* dg_step under DG_INTEGRATOR_LSERK4 (reading Q8) for callers that cannot allocate (CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same time loop, but the 2N-storage residual of the stage kernel lives in a
 * file-scope device array of the library instead of the workspace, and the call makes no cudaMalloc / cudaFree and uses no
 * allocating library routine.  Inputs and outputs are the context's bound workspace as for dg_step.  The array is
 * dg_static_scratch_bytes = 8 MiB on every GPU that loads the library, until the process exits; a state whose field
 * array [nslots][4 Np] is larger is rejected with DG_ERR_NOMEM (use dg_step).  DG_ERR_STATE unless the integrator is
 * LSERK4 and dg_set_profiling is off (profiling creates events).  The array is shared by all calls and contexts on a GPU
 * and keeps the last call's contents: every call clears what it uses first; calls whose kernels overlap on the GPU
 * (different streams) race on it - serialise them.  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress): make one call before capturing a graph. */
int dg_step_lserk4_static(dg_ctx* ctx, int nsteps);
int dg_static_scratch_bytes(size_t* n);
/* Prescribed-exterior faces (DG_BC_PRESCRIBED; plane-wave tests): exterior traces (p+, n.v+ with the
 * owner's outward normal) ext[nbnd][Nfp][2] in boundary-face-list order, used by every following
 * right-hand side until replaced.  Entries of faces of another type are ignored. */
int dg_set_exterior(dg_ctx* ctx, const double* ext);

/* ---- domain decomposition ---------------------------------------
 * A sub-domain is an ordinary ctx over its part of the mesh whose cut faces are DG_BC_PRESCRIBED faces.  Their exterior
 * state is the neighbouring sub-domain's exposed trace at the coinciding node, fetched on the DEVICE by dg_halo_pull
 * straight from the neighbour's trace buffer (its own ctx on this GPU, or a peer pointer over NVLink): no host staging.
 * dg_set_exterior_impedance: Zext[nbnd] = rho c of the element behind each boundary face (<= 0: none; NULL: clear), so
 *   that a halo face gets the same single-valued impedance (Z- + Z+) / 2 as the interior face it replaces (reading Q4);
 *   call before dg_workspace_bytes / dg_bind_workspace (it unbinds).
 * dg_get_slots: slot_of[K], the position of every element in the level-sorted device order (a trace record of face f
 *   of element k is record slot_of[k] * 4 + f of the trace buffer: p[Nfp] then n.v[Nfp], own face-node order on
 *   boundary faces).
 * dg_get_trace_device: device pointer / size of the buffer that holds the exposed traces at the current time (it
 *   alternates between two buffers from step to step: query it before every dg_halo_pull).
 * dg_set_halo: halo set `set` (0..31, one per neighbouring sub-domain and level of the elements behind the cut, filled
 *   in ascending order) of nh faces:
 *   bnd_index[nh] (boundary-face-list index here), src_record[nh] (record in that neighbour's buffer), src_pos[nh][Nfp]
 *   (position in that record of the node coinciding with my face node i).  After bind.
 * dg_halo_pull: enqueue the fetch of one set on this ctx's stream (the caller orders it after the neighbour's last step).
 * A time step of the decomposed single-rate problem = every sub-domain pulls, then every sub-domain takes dg_step(1).
 *
 * Multi-rate sub-domains (the paper partitions the multi-rate scheme, cell weights 2^(l-1)):
 * dg_set_model_levels: dg_set_model with the levels and the finest step of the WHOLE mesh imposed instead of derived from
 *   this part alone: level[K] (0 = coarsest; face neighbours at most one apart), dt_local = step of the finest level,
 *   bnd_level[nbnd] = level of the element behind each boundary face in the neighbouring sub-domain (-1: none; NULL: none
 *   anywhere) - an element whose neighbour across the cut is finer exposes half-step traces (eq (19)) like one whose finer
 *   neighbour is inside.
 * dg_step_fine: advance nfine FINE steps of the multi-rate cycle (Alg. 1; fine step m of a global step advances the
 *   levels whose step starts there); dg_step needs the scheme at the start of a global step.
 * dg_get_trace_levels: current[nlevels] = the buffer that holds, for the elements of level l, the exposed traces at the
 *   time level l has reached; half = the buffer of the half-step traces of the elements in mid-step; nbytes of each.
 * dg_halo_sources: the FUSED exchange - instead of dg_halo_pull launches, the step kernel itself (k_pipe / k_step, AB
 *   scheme) reads the exterior state of every halo face from the neighbour's trace buffer while it forms the penalties of
 *   that face: src_trace_device[nsets] = the source buffer of every halo set for the NEXT fine step (one dg_step(1) of a
 *   single-rate ctx or one dg_step_fine(1); consumed by it - the buffers alternate).  With peer pointers the loads cross
 *   NVLink inside the step kernel, block by block, overlapped with the other blocks' arithmetic; no k_halo launch, no
 *   exterior array in between.  The caller orders the step after the neighbours' previous step, and the neighbours' next
 *   step after this one (they overwrite the buffer two steps later).  DG_ERR_UNSUPPORTED for LSERK4 / DGRTM_KERNEL=tc.
 * Fine step m of the decomposed problem = every sub-domain pulls every set - from current[l] of the neighbour if the
 *   level l of the elements behind that set starts a step at m, else from its half-step buffer - then every sub-domain
 *   takes dg_step_fine(1) (paper_1506_00907_b200/decomp.py). */
int dg_set_exterior_impedance(dg_ctx* ctx, const double* Zext);
int dg_get_slots(dg_ctx* ctx, int64_t* slot_of);
int dg_get_trace_device(dg_ctx* ctx, void** dptr, size_t* nbytes);
int dg_set_halo(dg_ctx* ctx, int set, int64_t nh, const int32_t* bnd_index, const int64_t* src_record, const int32_t* src_pos);
int dg_halo_pull(dg_ctx* ctx, int set, const void* src_trace_device);
int dg_set_model_levels(dg_ctx* ctx, const double* rho, const double* c, int nlevels, double dt_local, const int32_t* level,
                        const int32_t* bnd_level);
int dg_step_fine(dg_ctx* ctx, int nfine);
int dg_get_trace_levels(dg_ctx* ctx, void** current /* [nlevels] */, void** half, size_t* nbytes);
int dg_halo_sources(dg_ctx* ctx, int nsets, const void* const* src_trace_device /* [nsets] */);
/* The three trace buffers of a wavefield (field 0: source / forward, 1: receivers - needs the RTM region): the two that
 * alternate as a level's current buffer, and the half-step buffer.  Sub-domains that step in lock-step alternate alike, so
 * a process exchanges these addresses ONCE and derives its neighbour's current buffer from its own (decomp.py). */
int dg_get_trace_buffers(dg_ctx* ctx, int field, void** buffers /* [3] */, size_t* nbytes);

/* ---- RTM (Fig. 1) ---------------------------------------------------
 * History = boundary traces (p, n.v) of every absorbing boundary face node at every right-hand-side
 * evaluation time of its owner plus the final time (layout reading Q12) - it stays in
 * HBM.  rtm_history_bytes: size for shots of nsteps global steps. */
int rtm_set_receiver_capacity(dg_ctx* ctx, int64_t max_receivers);   /* before rtm_history_bytes / rtm_bind_history */
int rtm_history_bytes(dg_ctx* ctx, int nsteps, size_t* n);
int rtm_bind_history(dg_ctx* ctx, void* dptr, size_t n);
/* Boundary-trace spill to host memory for histories larger than HBM (the paper keeps the traces in host RAM / on disk,
 * PAPER.md:399-407).  rtm_spill_bytes: host bytes of the whole trace history of shots of nsteps
 * global steps.  rtm_set_trace_spill: `host` = caller-owned PINNED host memory of n bytes (borrowed until replaced or
 * dg_destroy; NULL switches the spill off), `window` >= 2 = records of the coarsest level kept on the device (level l
 * keeps window << l): the RTM region then holds that ring only, every captured record is copied to the host on a second
 * stream behind the step that wrote it, and the backward phase fetches the records it replays window - 1 evaluations
 * ahead.  Call before rtm_history_bytes / rtm_bind_history (it unbinds the RTM region).  Results are bit-identical to
 * the in-HBM history. */
/* rtm_set_spill_packing(ctx, 1): the HOST copy of a spilled history keeps every value in half the bytes - fp64 -> fp32,
 * fp32 -> bf16 (relative rounding 2^-24 / 2^-8 per value; the paper names compression of the boundary data as future work,
 * PAPER.md:512).  Lossy: the reconstructed source wavefield and the image change at that level (documented with the
 * measured error in DESIGN.md); the device ring and every kernel of the step keep full precision, the conversion runs on
 * the copy stream; the replay takes EVERY record from the rounded copy (also those still in the ring), so one history
 * gives one result.  Call before rtm_spill_bytes / rtm_set_trace_spill / rtm_history_bytes (it unbinds the RTM region). */
int rtm_set_spill_packing(dg_ctx* ctx, int on);
int rtm_spill_bytes(dg_ctx* ctx, int nsteps, size_t* n);
int rtm_set_trace_spill(dg_ctx* ctx, void* host, size_t n, int window);
/* Forward phase: from rest at t = 0, source on, nsteps global steps; captures the boundary traces,
 * keeps q(t_f) on the device, records p(x_r, j dt_local), j = 0..nfine, into data_out[nr][nfine+1]
 * (host; may be NULL).  Synchronises. */
int rtm_forward_shot(dg_ctx* ctx, int nsteps, double* data_out);
/* Backward phase: source field reconstructed from q(t_f) with the stored traces as exterior states,
 * receiver field from rest with data[nr][nfine+1] injected (eq (15) weights), both stepped backward
 * in time with negative penalty parameters; before every update the step's
 * contribution to the image is accumulated with the AB-consistent integral (eqs (20)-(24) PAPER.md:
 * 174-204, corrected coefficients: reading Q1, sign: Q1b) of the classical (eq (4)) or
 * the characteristic pressure+velocity condition q_S^- q_R^+, q^+- = p +- c rho e.v (eqs (5)-(8)
 * PAPER.md:55-68), e = updir.  Only steps whose start index (forward numbering of global steps) is
 * > first_image_step contribute... i.e. imaging over t in [first_image_step*dt_global, t_f]
 * (PAPER.md:460).  Images of successive shots add up.  Synchronises. */
int rtm_backward_shot(dg_ctx* ctx, int nsteps, const double* data, const double updir[3],
                      int imaging, int64_t first_image_step);
/* A phase of a shot in PARTS - for a domain decomposition, where the sub-domains exchange halo traces between the fine
 * steps ("for the backward run ... both source and receivers simulations are performed using the same mesh
 * partition", so the imaging condition needs no exchange): fine steps [fine0, fine0 + nfine) of a phase of nsteps global
 * steps.  The part with fine0 = 0 initialises the phase exactly as the _shot call does (data / updir / imaging are read
 * then and on every part; data may be NULL after the first), the part that reaches nsteps * 2^(L-1) finishes it (final
 * capture and sample, data_out; earlier parts ignore data_out and do not synchronise).  An empty part at 0 (nfine = 0)
 * initialises alone - the trace buffers can then be asked for before the first step (a backward part at 0 that carries
 * signals always starts the phase anew).  The parts follow one another
 * (DG_ERR_STATE otherwise).  rtm_forward_shot(n, d) = rtm_forward_part(n, 0, n * 2^(L-1), d), likewise backward.
 * rtm_get_trace_levels: dg_get_trace_levels for field 0 (source wavefield) or 1 (receiver wavefield).
 * rtm_halo_sources: dg_halo_sources for the receiver wavefield; a two-field step needs both, each for ONE fine step. */
int rtm_forward_part(dg_ctx* ctx, int nsteps, int64_t fine0, int64_t nfine, double* data_out);
int rtm_backward_part(dg_ctx* ctx, int nsteps, const double* data, const double updir[3], int imaging,
                      int64_t first_image_step, int64_t fine0, int64_t nfine);
int rtm_get_trace_levels(dg_ctx* ctx, int field, void** current /* [nlevels] */, void** half, size_t* nbytes);
int rtm_halo_sources(dg_ctx* ctx, int nsets, const void* const* src_trace_device /* [nsets] */);
int rtm_image_read(dg_ctx* ctx, double* I_out /* [K][Np] */);
int rtm_image_zero(dg_ctx* ctx);
/* Device address and size of the image in the library's blocked layout [block][Np][32] (device precision), inside the
 * caller's history buffer.  For the one collective of a shot-per-GPU survey: replicas
 * that hold the same mesh and model share the layout, so their images add element-wise in place (e.g. one NCCL
 * all-reduce over a view of the caller's buffer); rtm_image_read then returns the stacked image.  Synchronises. */
int rtm_image_device(dg_ctx* ctx, void** dptr, size_t* nbytes);

/* ---- getters (parity checks; all synchronise) ----------------------------------------------------*/
int dg_get_sizes(const dg_ctx* ctx, int64_t* K, int* Np, int* Nfp, int64_t* nbnd, int64_t* nr);
int dg_get_nodes(const dg_ctx* ctx, double* r, double* s, double* t /* [Np] each */);
/* Dr,Ds,Dt [Np][Np]; LIFT [Np][4*Nfp] (column block f = L_f); Fmask [4][Nfp].  NULL = skip. */
int dg_get_operators(const dg_ctx* ctx, double* Dr, double* Ds, double* Dt, double* LIFT,
                     int32_t* Fmask);
/* EToE, EToF [K][4] (-1 on boundary faces); mapP [K][4][Nfp]: face-node index on the neighbour face
 * that coincides with face node i (identity on boundary faces).  NULL = skip. */
int dg_get_connectivity(const dg_ctx* ctx, int32_t* EToE, int32_t* EToF, int32_t* mapP);
/* Boundary-face list (ascending (k,f)): element, local face, type.  [nbnd] each, NULL = skip. */
int dg_get_boundary_faces(const dg_ctx* ctx, int32_t* bk, int32_t* bf, int32_t* bc);
/* J [K], ginv [K][3][3] (= d r_j / d x_i), normals [K][4][3], gsur [K][4], ell [K].  NULL = skip. */
int dg_get_geometry(const dg_ctx* ctx, double* J, double* ginv, double* normals, double* gsur,
                    double* ell);
int dg_get_levels(const dg_ctx* ctx, int32_t* level /* [K] */);
int dg_get_dt(const dg_ctx* ctx, double* dt_local, int* nlocal /* fine steps per global step */);
int dg_get_time(const dg_ctx* ctx, double* t);
int dg_get_source(const dg_ctx* ctx, int32_t* k, double* w /* [Np] */);
int dg_get_receivers(const dg_ctx* ctx, int32_t* k /* [nr] */, double* rows /* [nr][Np] */,
                     double* w /* [nr][Np] */);
int dg_get_fields(dg_ctx* ctx, double* q /* [K][4][Np] */);
/* Exposed traces qf[K][4][Nfp][2] = (p, n.v) in the OWNER's face-node order. */
int dg_get_traces(dg_ctx* ctx, double* qf);
/* Right-hand side of the current state at the current time, evaluated now by the volume kernel, the
 * surface kernel or both (no source term); r[K][4][Np].  Does not advance or disturb the state.
 * direction = +1 / -1 (sign of the penalty parameters). */
int dg_get_rhs(dg_ctx* ctx, int which, int direction, double* r);
/* RTM bookkeeping: per level, the boundary-face-list indices of the stored faces (ascending) and the
 * number of records.  faces may be NULL to query nfaces / nrecords only. */
int rtm_get_trace_index(const dg_ctx* ctx, int level, int64_t* nfaces, int64_t* nrecords,
                        int32_t* faces);
/* Record j of a level: buf[nfaces][Nfp][2] = (p, n.v). */
int rtm_get_traces(dg_ctx* ctx, int level, int64_t record, double* buf);
/* Wavefields kept by the RTM phases: which = 0 final forward state q(t_f), 1 = reconstructed source
 * field, 2 = receiver field (the latter two after rtm_backward_shot). */
int rtm_get_fields(dg_ctx* ctx, int which, double* q /* [K][4][Np] */);

/* ---- measurement ------------------------------------------------------------------------------
 * Counts of kernels launched by this ctx since creation (bench.py's gpu_launches). */
int dg_get_launch_count(const dg_ctx* ctx, int64_t* n);
/* Per-kernel timing.  dg_set_profiling(ctx, 1): every following kernel launch of this ctx is bracketed by
 * a CUDA event pair on the bound stream (adds ~2 us per launch; off by default).  dg_get_kernel_times
 * synchronises, sums the elapsed milliseconds and the launch counts per kernel class since the last
 * call into ms[DG_KC_COUNT], count[DG_KC_COUNT] and forgets the events. */
enum { DG_KC_RHS = 0, DG_KC_UPDATE, DG_KC_HALO, DG_KC_IMAGE_UPDATE, DG_KC_SOURCE, DG_KC_RECORD,
       DG_KC_INJECT, DG_KC_CAPTURE, DG_KC_RK, DG_KC_STEP, DG_KC_STEP_IMAGE, DG_KC_COUNT };
int dg_set_profiling(dg_ctx* ctx, int on);
int dg_get_kernel_times(dg_ctx* ctx, double* ms, int64_t* count);
/* Enqueue `reps` launches of one kernel over the whole mesh on the bound stream (state is disturbed:
 * for kernel timing only).  which: 0 volume, 1 surface, 2 fused volume+surface, 3 update (18),
 * 4 backward update with fused imaging (two wavefields). */
int dg_bench_kernel(dg_ctx* ctx, int which, int reps);

/* Plain-ALU ceilings of the device for the roofline (needs no ctx): a register-only fused-multiply-add
 * loop, kind 0 = fp32 FFMA, 1 = packed fp32x2 FFMA2, 2 = fp64 DFMA; dscratch = at least 4 bytes x 2048 x (SM count)
 * of device memory (never written in practice), timed with a CUDA event pair on the stream; *tflops = 2 flop per FMA. */
int dg_measure_fma(int kind, void* dscratch, size_t scratch_bytes, void* cuda_stream, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* DGRTM_H */
