// C ABI of libdgrtm, part 3: the time-stepping schedule of Algorithm 1 on the
// device kernels, forward or backward in time, one or two wavefields.
#include <algorithm>
#include <cmath>

#include "ctx.h"

namespace dgrtm {

namespace {

inline int lvl_blk_end(const Model& md, int l) { return md.lvl_blk0[l] + md.lvl_nblk[l]; }

PointArgs point_args(dg_ctx* c, const Field& F) {
  PointArgs p;
  std::memset(&p, 0, sizeof(p));
  p.q = F.q;
  for (int s = 0; s < 3; ++s) p.hist[s] = F.hist[s];
  for (int l = 0; l < kMaxLevels; ++l) p.cur[l] = F.cur[l];
  return p;
}

}  // namespace

// right-hand side of levels l0..l1-1 of field F into `out` (a full-size [nslots][4Np] array)
void launch_rhs(dg_ctx* c, Field& F, char* out, int l0, int l1, int mode, double dir, char* capture,
                const char* replay) {
  const Model& md = c->model;
  RhsArgs a;
  std::memset(&a, 0, sizeof(a));
  a.q = F.q; a.qf = F.qf; a.rhs = out; a.geo = c->geo; a.nbr = c->nbr;
  a.blk0 = md.lvl_blk0[l0]; a.nblk = lvl_blk_end(md, l1 - 1) - a.blk0;
  a.mode = mode; a.dir = dir; a.capture = capture; a.replay = replay;
  a.ext = c->has_ext ? c->ext : nullptr;
  a.ops = c->ops;
  if (a.nblk > 0) DG_LAUNCH(c, KC_RHS, c->kt->rhs(a, c->stream));
}

// Algorithm 1 on the fused step kernel: per fine step ONE launch advances every level that sits at the
// step start (right-hand side at t_start, update to t_start + dt_l, traces into the level's other buffer,
// half-step traces for finer neighbours); readers pick, per neighbour level, the buffer holding the traces
// at t_start: the level's current buffer if that level is also at t_start, else (a coarser level in
// mid-step) its half-step buffer (eq (19)).
void run_mrab(dg_ctx* c, int nglobal, const RunOpts& o) {
  const Model& md = c->model;
  const int L = md.nlevels, nloc = c->nlocal, dir = o.direction;
  const double dtl = c->dt_local;
  if (c->has_prescribed && !c->has_ext) throw ApiError(DG_ERR_STATE, "prescribed-exterior faces need dg_set_exterior");
  if (o.nfields == 2 && !c->hist_bound) throw ApiError(DG_ERR_STATE, "two wavefields need the RTM region");
  int stride[kMaxLevels];
  for (int l = 0; l < L; ++l) stride[l] = 1 << (L - 1 - l);
  const int src_level = c->has_src ? md.level[c->src_k] : -1;
  const int64_t nsamp = (int64_t)c->hist_nsteps * nloc + 1;
  // p(x_r) at fine time m BEFORE the launch of fine step m: a level at its step start holds q(t); a level
  // in mid-step already holds q at the END of its step: p(t) = q_end - dt_l sum_s (a_s - I_s(theta)) r_s
  // with the interpolant (22) (reading Q13)
  auto sample_receivers = [&](int64_t m, int64_t jabs) {
    PointArgs p = point_args(c, *o.fields[0]);
    p.nr = (int)c->nr; p.rcv_slot = c->d_rcv_slot; p.rcv_row = c->d_rcv_row; p.rcv_level = c->d_rcv_level;
    p.data = c->d_data; p.nsamp = nsamp; p.sample = jabs;
    for (int l = 0; l < L; ++l) {
      const int off = (int)((m + o.fine_phase) % stride[l]);
      if (!off) continue;
      const int order = o.fields[0]->nhist[l];
      double w[3] = {0, 0, 0};
      ab_partial(order, (double)off / stride[l], w);
      const AbCoef& co = ab_coef(order);
      for (int s = 0; s < 3; ++s) p.lw[l][s] = -dir * stride[l] * dtl * (co.a[s] - w[s]);
    }
    DG_LAUNCH(c, KC_RECORD, c->kt->record(p, c->stream));
  };

  StepArgs a;
  std::memset(&a, 0, sizeof(a));
  a.nfields = o.nfields; a.nlevels = L;
  a.geo = c->geo; a.nbr = c->nbr; a.wperm = c->wperm; a.blkflag = c->d_blkflag;
  a.ext = c->has_ext ? c->ext : nullptr;
  if (c->halo_src_valid) {   // fused halo exchange: this call's launches read the neighbours' buffers
    if ((o.nfine >= 0 ? o.nfine : (int64_t)nglobal * nloc) != 1)
      throw ApiError(DG_ERR_STATE, "dg_halo_sources serves ONE fine step (the trace buffers alternate): dg_step(1) single-rate, dg_step_fine(1)");
    const size_t nbf = c->mesh.bnd_k.size();
    a.halo_rec = reinterpret_cast<const long long*>(c->d_halo_face);
    a.halo_set = reinterpret_cast<const int*>(c->d_halo_face + nbf * 8);
    a.halo_pos = reinterpret_cast<const int*>(c->d_halo_face + nbf * 12);
    for (int x = 0; x < kMaxHaloSets; ++x) a.halo_src[x] = c->halo_src[x];
    if (o.nfields == 2) {
      if (!c->halo_src2_valid) throw ApiError(DG_ERR_STATE, "two wavefields: rtm_halo_sources must name the receiver field's sources too");
      for (int x = 0; x < kMaxHaloSets; ++x) a.halo_src2[x] = c->halo_src2[x];
    }
    c->halo_src2_valid = false;
    c->halo_src_valid = false;                 // the buffers alternate: sources are good for the step they were given for
  }
  a.sched = sched_counters(c);
  a.sched_mode = L > 1 ? 1 : 0;     // blocks of a multi-rate launch differ in cost and sit sorted by level
  a.dir = (double)dir;
  a.ops = c->ops; a.ops.D3T = c->d_D3P; a.ops.LIFTT = c->d_LTP;
  a.ops2_D3Q = c->d_D3Q; a.ops2_LTQ = c->d_LTQ;
  const bool pipe = c->use_pipe && c->kt->pipe != nullptr && c->ops.nperm <= 8;   // (a triangle has 6; the pipelined kernel's gather table holds 8)
  const bool tc = c->use_tc && c->kt->tc != nullptr && o.nfields == 1;
  a.image = c->image; a.img_scratch = c->scratch; a.characteristic = (o.imaging & 1) != 0;
  a.trapezoid = (o.imaging & 2) != 0;
  for (int d = 0; d < 3; ++d) a.e[d] = o.updir[d];
  for (int fi = 0; fi < o.nfields; ++fi) {
    a.q[fi] = o.fields[fi]->q;
    if (o.source_on[fi]) { a.pt_index[fi] = c->d_pt_src; a.pt_val[fi] = c->d_src_w; }
    if (o.inject_field == fi && !c->grp_slot.empty()) { a.pt_index[fi] = c->d_pt_rcv; a.pt_val[fi] = c->d_pt_val; a.pt_scale[fi] = 1.0; }
  }
  for (int l = 0; l < L; ++l) a.lv[l].blk_end = md.lvl_blk0[l] + md.lvl_nblk[l];

  const int64_t nfine = o.nfine >= 0 ? o.nfine : (int64_t)nglobal * nloc;
  for (int64_t m = 0; m < nfine; ++m) {
    const int64_t jabs = o.first_fine + dir * m;
    const double t_start = o.t0 + dir * (double)m * dtl;
    if (o.record && c->nr > 0) sample_receivers(m, jabs);
    if (o.inject_field >= 0 && !c->grp_slot.empty()) {     // injection amounts of this fine step (eq (15))
      PointArgs p = point_args(c, *o.fields[o.inject_field]);
      p.rcv_w = c->d_rcv_w; p.data = c->d_data; p.nsamp = nsamp; p.sample = jabs;
      p.g0 = 0; p.ng = (int)c->grp_slot.size();
      p.grp_slot = c->d_grp_slot; p.grp_off = c->d_grp_off; p.grp_rcv = c->d_grp_rcv; p.pt_out = c->d_pt_val;
      DG_LAUNCH(c, KC_INJECT, c->kt->inject(p, c->stream));
    }
    int lmin = L - 1;
    while (lmin > 0 && (m + o.fine_phase) % stride[lmin - 1] == 0) --lmin;   // strides are powers of two
    for (int l = 0; l < L; ++l) {
      StepLevel& S = a.lv[l];
      const bool active = l >= lmin;
      S.active = active;
      for (int fi = 0; fi < o.nfields; ++fi) {
        Field& F = *o.fields[fi];
        // traces at t_start: the current buffer of a level that is at t_start, the half-step buffer otherwise
        S.qf_read[fi] = active ? F.qfb[F.par[l]] : F.qfh;
        if (!active) continue;
        F.cur[l] = (F.cur[l] + 1) % 3;
        F.nhist[l] = std::min(F.nhist[l] + 1, 3);
        S.r0[fi] = F.hist[F.cur[l]]; S.r1[fi] = F.h(l, 1); S.r2[fi] = F.h(l, 2);
        S.qf_write[fi] = F.qfb[F.par[l] ^ 1];
        S.qf_half[fi] = (l + 1 < L && !md.coarse_nb[l].empty()) ? F.qfh : nullptr;
      }
      if (!active) continue;
      const AbCoef& co = ab_coef(o.fields[0]->nhist[l]);
      const double dts = dir * (double)stride[l] * dtl;
      S.dts = dts;
      for (int s = 0; s < 3; ++s) { S.c[s] = dts * co.a[s]; S.d[s] = dts * (co.b[s] - co.a[s]); S.abar[s] = co.abar[s]; }
      for (int s = 0; s < 9; ++s) S.C[s] = co.C[s];
      const bool stored = !md.stored[l].empty();
      S.capture = (o.capture && stored) ? record_ptr(c, l, jabs / stride[l]) : nullptr;
      S.replay = (o.replay && stored) ? record_ptr(c, l, jabs / stride[l]) : nullptr;
      if (S.capture) spill_before_capture(c, l, jabs / stride[l]);
      if (S.replay) spill_before_replay(c, l, jabs / stride[l]);
      const int64_t jlast = jabs + dir * (stride[l] - 1);   // start of the fine step on which this update lands
      S.image_on = o.image && std::min(jlast, jlast + dir) >= o.image_min_fine;
    }
    for (int fi = 0; fi < o.nfields; ++fi)
      if (o.source_on[fi]) a.pt_scale[fi] = (src_level >= lmin) ? ricker(t_start, c->f0, c->tp, c->amp) : 0.0;
    a.blk0 = md.lvl_blk0[lmin];
    a.nblk = (int)md.nblocks - a.blk0;
    if (a.nblk > 0) {
      if (pipe && (o.nfields == 2 || !tc)) { a.sched_sel = c->sched_sel; c->sched_sel ^= 1; a.reverse = L == 1 ? (int)(m & 1) : 0; }   // only launches that take tickets flip the counters
      if (o.nfields == 2) DG_LAUNCH(c, KC_STEP_IMAGE, pipe ? c->kt->pipe2(a, c->stream) : c->kt->step2(a, c->stream));
      else DG_LAUNCH(c, KC_STEP, tc ? c->kt->tc(a, c->stream) : (pipe ? c->kt->pipe(a, c->stream) : c->kt->step(a, c->stream)));
    }
    for (int l = lmin; l < L; ++l) {
      if (a.lv[l].capture) spill_after_capture(c, l, jabs / stride[l]);
      if (a.lv[l].replay) spill_after_replay(c, l, jabs / stride[l]);
      for (int fi = 0; fi < o.nfields; ++fi) o.fields[fi]->par[l] ^= 1;
    }
  }
  const int64_t jend = o.first_fine + dir * nfine;
  if (!o.finish) return;
  if (o.capture) {
    for (int l = 0; l < L; ++l) {
      if (md.stored[l].empty()) continue;
      CaptureArgs ca;
      std::memset(&ca, 0, sizeof(ca));
      ca.q = o.fields[0]->q; ca.geo = c->geo; ca.faces = c->d_stored[l]; ca.nfaces = (int)md.stored[l].size();
      ca.record = record_ptr(c, l, jend / stride[l]); ca.ops = c->ops;
      spill_before_capture(c, l, jend / stride[l]);
      DG_LAUNCH(c, KC_CAPTURE, c->kt->capture(ca, c->stream));
      spill_after_capture(c, l, jend / stride[l]);
    }
  }
  if (o.record && c->nr > 0) sample_receivers(0, jend);
}

// five-stage LSERK4 of Carpenter & Kennedy (not in the paper; BASELINE.json config 1, reading Q8)
void run_lserk4(dg_ctx* c, int nsteps) {
  static const double A[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                              -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
  static const double B[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                              1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                              2277821191437.0 / 14882151754819.0};
  static const double C[5] = {0.0, 1432997174477.0 / 9575080441755.0, 2526269341429.0 / 6820363962896.0,
                              2006345519317.0 / 3224310063776.0, 2802321613138.0 / 2924317926251.0};
  const Model& md = c->model;
  if (md.nlevels != 1) throw ApiError(DG_ERR_UNSUPPORTED, "LSERK4 is single-rate only");
  if (c->has_prescribed && !c->has_ext) throw ApiError(DG_ERR_STATE, "prescribed-exterior faces need dg_set_exterior");
  Field& F = c->F;
  normalize_traces(c, F);
  const double dt = c->dt_local;
  for (int n = 0; n < nsteps; ++n) {
    const double t = c->t0 + (double)(c->fine + n) * dt;
    for (int st = 0; st < 5; ++st) {
      char* r = F.hist[0];
      launch_rhs(c, F, r, 0, 1, RHS_VOL | RHS_SURF, 1.0, nullptr, nullptr);
      if (c->has_src) {
        PointArgs p;
        std::memset(&p, 0, sizeof(p));
        p.rhs = r; p.src_slot = (int)md.slot_of[c->src_k]; p.src_w = c->d_src_w;
        p.amp_now = ricker(t + C[st] * dt, c->f0, c->tp, c->amp);
        DG_LAUNCH(c, KC_SOURCE, c->kt->source(p, c->stream));
      }
      RkArgs k;
      std::memset(&k, 0, sizeof(k));
      k.q = F.q; k.qf = F.qf; k.res = c->scratch; k.r = r; k.geo = c->geo; k.wperm = c->wperm;
      k.blk0 = 0; k.nblk = (int)md.nblocks; k.A = A[st]; k.B = B[st]; k.dt = dt; k.ops = c->ops;
      DG_LAUNCH(c, KC_RK, c->kt->rk(k, c->stream));
    }
  }
}

}  // namespace dgrtm

using namespace dgrtm;

extern "C" {

int dg_step(dg_ctx* ctx, int nsteps) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (nsteps < 0) throw ApiError(DG_ERR_ARG, "nsteps must be >= 0");
  if (ctx->integrator == DG_INTEGRATOR_LSERK4) {
    run_lserk4(ctx, nsteps);
    ctx->fine += nsteps;
  } else {
    if (ctx->fine % ctx->nlocal) throw ApiError(DG_ERR_STATE, "dg_step_fine left the scheme inside a global step: finish it first");
    RunOpts o;
    o.direction = 1; o.fields[0] = &ctx->F; o.nfields = 1; o.source_on[0] = ctx->has_src;
    o.first_fine = ctx->fine; o.t0 = ctx->t0 + (double)ctx->fine * ctx->dt_local;
    run_mrab(ctx, nsteps, o);
    ctx->fine += (int64_t)nsteps * ctx->nlocal;
  }
  check_launches(ctx);
  DG_CATCH(ctx)
}

int dg_step_fine(dg_ctx* ctx, int nfine) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (nfine < 0) throw ApiError(DG_ERR_ARG, "nfine must be >= 0");
  if (ctx->integrator != DG_INTEGRATOR_AB3) throw ApiError(DG_ERR_STATE, "dg_step_fine advances the multi-rate AB scheme");
  RunOpts o;
  o.direction = 1; o.fields[0] = &ctx->F; o.nfields = 1; o.source_on[0] = ctx->has_src;
  o.first_fine = ctx->fine; o.t0 = ctx->t0 + (double)ctx->fine * ctx->dt_local;
  o.fine_phase = ctx->fine % ctx->nlocal; o.nfine = nfine;
  run_mrab(ctx, 0, o);
  ctx->fine += nfine;
  check_launches(ctx);
  DG_CATCH(ctx)
}

int dg_get_rhs(dg_ctx* ctx, int which, int direction, double* r) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!r) throw ApiError(DG_ERR_ARG, "r is NULL");
  if (direction != 1 && direction != -1) throw ApiError(DG_ERR_ARG, "direction must be +1 or -1");
  if (ctx->has_prescribed && !ctx->has_ext) throw ApiError(DG_ERR_STATE, "prescribed-exterior faces need dg_set_exterior");
  int mode;
  switch (which) {
    case DG_RHS_VOLUME: mode = RHS_VOL; break;
    case DG_RHS_SURFACE: mode = RHS_SURF; break;
    case DG_RHS_TOTAL: mode = RHS_VOL | RHS_SURF; break;
    default: throw ApiError(DG_ERR_ARG, "which must be DG_RHS_VOLUME, DG_RHS_SURFACE or DG_RHS_TOTAL");
  }
  // the scratch array doubles as the LSERK4 residual, which is dead between steps (A_1 = 0)
  cuda_check(cudaMemsetAsync(ctx->scratch, 0, field_bytes(ctx), ctx->stream), "memset scratch");
  normalize_traces(ctx, ctx->F);
  launch_rhs(ctx, ctx->F, ctx->scratch, 0, ctx->model.nlevels, mode, (double)direction, nullptr, nullptr);
  check_launches(ctx);
  fields_from_device(ctx, r, ctx->scratch);
  DG_CATCH(ctx)
}

int dg_get_launch_count(const dg_ctx* ctx, int64_t* n) {
  if (!ctx || !n) return DG_ERR_ARG;
  *n = ctx->launches;
  return DG_OK;
}

int dg_set_profiling(dg_ctx* ctx, int on) {
  DG_TRY(ctx)
  ctx->prof = on != 0;
  DG_CATCH(ctx)
}

int dg_get_kernel_times(dg_ctx* ctx, double* ms, int64_t* count) {
  DG_TRY(ctx)
  if (!ms || !count) throw ApiError(DG_ERR_ARG, "ms / count is NULL");
  if (ctx->bound) sync_stream(ctx);
  for (int k = 0; k < KC_COUNT; ++k) { ms[k] = 0; count[k] = 0; }
  for (ProfEvent& e : ctx->prof_ev) {
    float t = 0;
    cuda_check(cudaEventElapsedTime(&t, e.a, e.b), "cudaEventElapsedTime");
    ms[e.cls] += t; count[e.cls]++;
    cudaEventDestroy(e.a); cudaEventDestroy(e.b);
  }
  ctx->prof_ev.clear();
  DG_CATCH(ctx)
}

int dg_bench_kernel(dg_ctx* ctx, int which, int reps) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (reps < 0) throw ApiError(DG_ERR_ARG, "reps must be >= 0");
  const Model& md = ctx->model;
  Field& F = ctx->F;
  normalize_traces(ctx, F);
  for (int i = 0; i < reps; ++i) {
    switch (which) {
      case 0: launch_rhs(ctx, F, F.hist[0], 0, md.nlevels, RHS_VOL, 1.0, nullptr, nullptr); break;
      case 1: launch_rhs(ctx, F, F.hist[0], 0, md.nlevels, RHS_SURF, 1.0, nullptr, nullptr); break;
      case 2: launch_rhs(ctx, F, F.hist[0], 0, md.nlevels, RHS_VOL | RHS_SURF, 1.0, nullptr, nullptr); break;
      case 3: {
        UpdateArgs u;
        std::memset(&u, 0, sizeof(u));
        u.q = F.q; u.qf = F.qf; u.h0 = F.hist[0]; u.h1 = F.hist[1]; u.h2 = F.hist[2];
        u.geo = ctx->geo; u.wperm = ctx->wperm; u.blk0 = 0; u.nblk = (int)md.nblocks;
        u.c0 = 1e-30; u.c1 = -1e-30; u.c2 = 1e-30; u.ops = ctx->ops;
        DG_LAUNCH(ctx, KC_UPDATE, ctx->kt->update(u, ctx->stream));
        break;
      }
      case 4: {
        if (!ctx->hist_bound) throw ApiError(DG_ERR_STATE, "rtm_bind_history first");
        ImageArgs a;
        std::memset(&a, 0, sizeof(a));
        Field& R = ctx->R;
        a.qS = F.q; a.qfS = F.qf; a.hS0 = F.hist[0]; a.hS1 = F.hist[1]; a.hS2 = F.hist[2];
        a.qR = R.q; a.qfR = R.qf; a.hR0 = R.hist[0]; a.hR1 = R.hist[1]; a.hR2 = R.hist[2];
        a.image = ctx->image; a.geo = ctx->geo; a.wperm = ctx->wperm; a.blk0 = 0; a.nblk = (int)md.nblocks;
        a.dts = -1e-30;
        const AbCoef& co = ab_coef(3);
        for (int s = 0; s < 3; ++s) { a.a[s] = co.a[s]; a.abar[s] = co.abar[s]; }
        for (int s = 0; s < 9; ++s) a.C[s] = co.C[s];
        a.e[2] = -1; a.characteristic = 1; a.ops = ctx->ops;
        DG_LAUNCH(ctx, KC_IMAGE, ctx->kt->image_update(a, ctx->stream));
        break;
      }
      default: throw ApiError(DG_ERR_ARG, "which must be 0..4");
    }
  }
  check_launches(ctx);
  DG_CATCH(ctx)
}

}  // extern "C"
