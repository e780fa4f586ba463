// C ABI of libdgrtm, part 4: reverse-time migration (Fig. 1): forward
// phase with boundary-trace capture, backward phase with trace replay, receiver injection and the
// imaging condition fused into the update.  All history stays in HBM (PAPER.md:407 kept it on the
// host / HDD because a K20 could not hold it).
#include <algorithm>
#include <map>

#include "ctx.h"

using namespace dgrtm;

namespace {

int64_t records_of_level(const dg_ctx* c, int l, int nsteps) { return ((int64_t)nsteps << l) + 1; }
// records of level l the DEVICE holds: all of them, or a ring of spill_window << l when the history spills to the host
int64_t device_records(const dg_ctx* c, int l, int nsteps) {
  const int64_t all = records_of_level(c, l, nsteps);
  return c->spill_window > 0 ? std::min<int64_t>(all, (int64_t)c->spill_window << l) : all;
}
size_t record_bytes(const dg_ctx* c, int l) { return c->model.stored[l].size() * (size_t)c->REC * c->rs; }
// bytes of one record in the host copy: as on the device, or every value in half the bytes (rtm_set_spill_packing)
size_t host_record_bytes(const dg_ctx* c, int l) { return c->spill_packed ? record_bytes(c, l) / 2 : record_bytes(c, l); }
size_t spill_host_bytes(const dg_ctx* c, int nsteps) {
  size_t n = 0;
  for (int l = 0; l < c->model.nlevels; ++l) n += ((size_t)records_of_level(c, l, nsteps) * host_record_bytes(c, l) + 255) / 256 * 256;
  return n;
}
void spill_release(dg_ctx* c) {
  for (int l = 0; l < kMaxLevels; ++l) {
    for (cudaEvent_t e : c->ev_step[l]) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_copy[l]) cudaEventDestroy(e);
    c->ev_step[l].clear(); c->ev_copy[l].clear(); c->slot_rec[l].clear();
  }
}
// ring bookkeeping of a bound history: which record every slot holds, one event pair per slot
void spill_setup(dg_ctx* c, int nsteps) {
  spill_release(c);
  if (c->spill_window <= 0) return;
  if (!c->copy_stream) cuda_check(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking), "cudaStreamCreate (trace spill)");
  size_t off = 0;
  for (int l = 0; l < c->model.nlevels; ++l) {
    c->hrec[l] = c->spill_host + off;
    off += ((size_t)records_of_level(c, l, nsteps) * host_record_bytes(c, l) + 255) / 256 * 256;
    const int64_t W = device_records(c, l, nsteps);
    c->slot_rec[l].assign((size_t)W, -1);
    c->ev_step[l].resize((size_t)W); c->ev_copy[l].resize((size_t)W);
    for (int64_t x = 0; x < W; ++x) {
      cuda_check(cudaEventCreateWithFlags(&c->ev_step[l][x], cudaEventDisableTiming), "cudaEventCreate");
      cuda_check(cudaEventCreateWithFlags(&c->ev_copy[l][x], cudaEventDisableTiming), "cudaEventCreate");
      cudaEventRecord(c->ev_copy[l][x], c->copy_stream);      // "no transfer pending"
    }
  }
}

void group_receivers(dg_ctx* c) {
  const Model& md = c->model;
  std::map<int64_t, std::vector<int32_t>> by_slot;
  for (int64_t r = 0; r < c->nr; ++r) by_slot[md.slot_of[c->rcv_k[r]]].push_back((int32_t)r);
  c->grp_slot.clear(); c->grp_off.assign(1, 0); c->grp_rcv.clear();
  for (auto& kv : by_slot) {
    c->grp_slot.push_back((int32_t)kv.first);
    for (int32_t r : kv.second) c->grp_rcv.push_back(r);
    c->grp_off.push_back((int32_t)c->grp_rcv.size());
  }
  // groups are ascending in slot, hence in level
  size_t g = 0;
  for (int l = 0; l <= md.nlevels; ++l) {
    const int64_t first_slot = l < md.nlevels ? (int64_t)md.lvl_blk0[l] * 32 : md.nslots;
    while (g < c->grp_slot.size() && c->grp_slot[g] < first_slot) ++g;
    c->grp_lvl0[l] = (int)g;
  }
  for (int l = md.nlevels + 1; l <= kMaxLevels; ++l) c->grp_lvl0[l] = (int)c->grp_slot.size();
}

void carve_history(dg_ctx* c, Carver& cv, int nsteps) {
  const Model& md = c->model;
  const size_t rs = c->rs;
  const int Np = c->Np;
  for (int l = 0; l < md.nlevels; ++l)
    c->rec[l] = cv.take((size_t)device_records(c, l, nsteps) * md.stored[l].size() * c->REC * rs);
  c->pack_stage = nullptr;
  if (c->spill_window > 0 && c->spill_packed) {   // staging of one packed record (the largest level's)
    size_t mx = 0;
    for (int l = 0; l < md.nlevels; ++l) mx = std::max(mx, record_bytes(c, l) / 2);
    c->pack_stage = cv.take(std::max<size_t>(mx, 16));
  }
  const size_t nr = (size_t)std::max<int64_t>(1, std::max(c->nr, c->nr_reserve));   // receiver capacity
  c->d_data = cv.take(nr * ((size_t)nsteps * c->nlocal + 1) * rs);
  c->d_rcv_slot = (int*)cv.take(nr * 4);
  c->d_rcv_level = (int*)cv.take(nr * 4);
  c->d_rcv_row = cv.take(nr * Np * rs);
  c->d_rcv_w = cv.take(nr * Np * rs);
  c->d_grp_slot = (int*)cv.take(nr * 4);
  c->d_grp_off = (int*)cv.take((nr + 1) * 4);
  c->d_grp_rcv = (int*)cv.take(nr * 4);
  c->R.q = cv.take(field_bytes(c));
  for (int s = 0; s < 3; ++s) c->R.hist[s] = cv.take(field_bytes(c));
  c->R.qf = cv.take(trace_bytes(c));
  c->R.qfb[0] = c->R.qf;
  c->R.qfb[1] = cv.take(trace_bytes(c));
  c->R.qfh = cv.take(trace_bytes(c));
  c->d_pt_rcv = (int*)cv.take((size_t)md.nslots * 4);
  c->d_pt_val = cv.take(nr * Np * rs);
  c->image = cv.take((size_t)md.nblocks * Np * 32 * rs);
  c->qfinal = cv.take(field_bytes(c));
}

struct HistPtrs {   // everything carve_history writes, for save / restore around a size query
  char* rec[kMaxLevels]; char* d_data; int* a; int* b; char* cc; char* d; int* e; int* f; int* g; Field R; char* image; char* qfinal; int* ptr; char* ptv; char* stage;
  void save(const dg_ctx* c) {
    for (int l = 0; l < kMaxLevels; ++l) rec[l] = c->rec[l];
    d_data = c->d_data; a = c->d_rcv_slot; b = c->d_rcv_level; cc = c->d_rcv_row; d = c->d_rcv_w;
    e = c->d_grp_slot; f = c->d_grp_off; g = c->d_grp_rcv; R = c->R; image = c->image; qfinal = c->qfinal;
    ptr = c->d_pt_rcv; ptv = c->d_pt_val; stage = c->pack_stage;
  }
  void restore(dg_ctx* c) const {
    for (int l = 0; l < kMaxLevels; ++l) c->rec[l] = rec[l];
    c->d_data = d_data; c->d_rcv_slot = a; c->d_rcv_level = b; c->d_rcv_row = cc; c->d_rcv_w = d;
    c->d_grp_slot = e; c->d_grp_off = f; c->d_grp_rcv = g; c->R = R; c->image = image; c->qfinal = qfinal;
    c->d_pt_rcv = ptr; c->d_pt_val = ptv; c->pack_stage = stage;
  }
};

void require_history(dg_ctx* c) {
  require_bound(c);
  if (!c->hist_bound) throw ApiError(DG_ERR_STATE, "no RTM history bound (rtm_history_bytes, rtm_bind_history)");
}

// host [nr][ncol_host] <-> device [nr][nsamp] (leading columns)
void copy_data(dg_ctx* c, double* host, const double* host_in, int64_t ncol) {
  const int64_t nsamp = (int64_t)c->hist_nsteps * c->nlocal + 1;
  const size_t rs = c->rs;
  if (c->nr == 0) return;
  const size_t n = (size_t)c->nr * ncol;
  char* tmp = host_stage(c, n * rs);             // pinned staging, conversions on host threads
  const bool f64 = c->precision == 64;
  if (host_in) {
    parallel_range(n, [&](size_t a, size_t b) {
      if (f64) for (size_t i = a; i < b; ++i) ((double*)tmp)[i] = host_in[i];
      else for (size_t i = a; i < b; ++i) ((float*)tmp)[i] = (float)host_in[i];
    });
    cuda_check(cudaMemcpy2DAsync(c->d_data, nsamp * rs, tmp, ncol * rs, ncol * rs, c->nr,
                                 cudaMemcpyHostToDevice, c->stream), "cudaMemcpy2DAsync data H2D");
    sync_stream(c);
  } else {
    cuda_check(cudaMemcpy2DAsync(tmp, ncol * rs, c->d_data, nsamp * rs, ncol * rs, c->nr,
                                 cudaMemcpyDeviceToHost, c->stream), "cudaMemcpy2DAsync data D2H");
    sync_stream(c);
    parallel_range(n, [&](size_t a, size_t b) {
      if (f64) for (size_t i = a; i < b; ++i) host[i] = ((const double*)tmp)[i];
      else for (size_t i = a; i < b; ++i) host[i] = (double)((const float*)tmp)[i];
    });
  }
}

}  // namespace

namespace dgrtm {
char* record_ptr(dg_ctx* c, int l, int64_t j) {
  const int64_t slot = c->spill_window > 0 ? j % (int64_t)c->slot_rec[l].size() : j;
  return c->rec[l] + (size_t)slot * record_bytes(c, l);
}
// forward: the slot of record j may be overwritten once its previous occupant has reached the host
void spill_before_capture(dg_ctx* c, int l, int64_t j) {
  if (c->spill_window <= 0) return;
  const size_t slot = (size_t)(j % (int64_t)c->slot_rec[l].size());
  cuda_check(cudaStreamWaitEvent(c->stream, c->ev_copy[l][slot], 0), "cudaStreamWaitEvent");
  c->slot_rec[l][slot] = j;
}
// forward: record j is complete when the launch that captured it is: send it to the host behind the compute stream
void spill_after_capture(dg_ctx* c, int l, int64_t j) {
  if (c->spill_window <= 0) return;
  const size_t slot = (size_t)(j % (int64_t)c->slot_rec[l].size()), nb = record_bytes(c, l);
  cuda_check(cudaEventRecord(c->ev_step[l][slot], c->stream), "cudaEventRecord");
  cuda_check(cudaStreamWaitEvent(c->copy_stream, c->ev_step[l][slot], 0), "cudaStreamWaitEvent");
  if (c->spill_packed) {   // pack on the copy stream into the staging record (stream order keeps it free), copy half the bytes
    launch_trace_pack(c->rec[l] + slot * nb, c->pack_stage, nb / c->rs, c->precision, c->copy_stream);
    cuda_check(cudaMemcpyAsync(c->hrec[l] + (size_t)j * (nb / 2), c->pack_stage, nb / 2, cudaMemcpyDeviceToHost, c->copy_stream), "packed trace record D2H");
    c->slot_rec[l][slot] = -1;   // the replay takes every record from the (rounded) host copy, also the last W: one result per history
  } else {
    cuda_check(cudaMemcpyAsync(c->hrec[l] + (size_t)j * nb, c->rec[l] + slot * nb, nb, cudaMemcpyDeviceToHost, c->copy_stream), "trace record D2H");
  }
  cuda_check(cudaEventRecord(c->ev_copy[l][slot], c->copy_stream), "cudaEventRecord");
}
namespace {
// make record j of level l resident in its ring slot (no-op if it is there or on its way); the bound stream does not wait
void spill_fetch(dg_ctx* c, int l, int64_t j) {
  const size_t slot = (size_t)(j % (int64_t)c->slot_rec[l].size()), nb = record_bytes(c, l);
  if (c->slot_rec[l][slot] == j) return;
  cuda_check(cudaStreamWaitEvent(c->copy_stream, c->ev_step[l][slot], 0), "cudaStreamWaitEvent");   // its last reader is done
  if (c->spill_packed) {
    cuda_check(cudaMemcpyAsync(c->pack_stage, c->hrec[l] + (size_t)j * (nb / 2), nb / 2, cudaMemcpyHostToDevice, c->copy_stream), "packed trace record H2D");
    launch_trace_unpack(c->pack_stage, c->rec[l] + slot * nb, nb / c->rs, c->precision, c->copy_stream);
  } else {
    cuda_check(cudaMemcpyAsync(c->rec[l] + slot * nb, c->hrec[l] + (size_t)j * nb, nb, cudaMemcpyHostToDevice, c->copy_stream), "trace record H2D");
  }
  cuda_check(cudaEventRecord(c->ev_copy[l][slot], c->copy_stream), "cudaEventRecord");
  c->slot_rec[l][slot] = j;
}
}  // namespace
// backward: record j must be in its slot before the launch that replays it
void spill_before_replay(dg_ctx* c, int l, int64_t j) {
  if (c->spill_window <= 0) return;
  spill_fetch(c, l, j);
  const size_t slot = (size_t)(j % (int64_t)c->slot_rec[l].size());
  cuda_check(cudaStreamWaitEvent(c->stream, c->ev_copy[l][slot], 0), "cudaStreamWaitEvent");
}
// backward: the launch that replayed record j is queued; its slot's next occupant, and the records the coming launches
// need, are fetched behind it (the ring keeps W - 1 records ahead of the replay)
void spill_after_replay(dg_ctx* c, int l, int64_t j) {
  if (c->spill_window <= 0) return;
  const int64_t W = (int64_t)c->slot_rec[l].size();
  const size_t slot = (size_t)(j % W);
  cuda_check(cudaEventRecord(c->ev_step[l][slot], c->stream), "cudaEventRecord");
  for (int64_t k = 1; k < W; ++k) { if (j - k < 0) break; spill_fetch(c, l, j - k); }
}
void upload_receiver_tables(dg_ctx* ctx) {
  group_receivers(ctx);
  const int64_t nr = ctx->nr;
  if (nr) {
    std::vector<int32_t> slot(nr), lvl(nr);
    for (int64_t r = 0; r < nr; ++r) {
      slot[r] = (int32_t)ctx->model.slot_of[ctx->rcv_k[r]];
      lvl[r] = ctx->model.level[ctx->rcv_k[r]];
    }
    upload_raw(ctx, ctx->d_rcv_slot, slot.data(), nr * 4);
    upload_raw(ctx, ctx->d_rcv_level, lvl.data(), nr * 4);
    upload_real(ctx, ctx->d_rcv_row, ctx->rcv_row.data(), ctx->rcv_row.size());
    upload_real(ctx, ctx->d_rcv_w, ctx->rcv_w.data(), ctx->rcv_w.size());
    upload_raw(ctx, ctx->d_grp_slot, ctx->grp_slot.data(), ctx->grp_slot.size() * 4);
    upload_raw(ctx, ctx->d_grp_off, ctx->grp_off.data(), ctx->grp_off.size() * 4);
    upload_raw(ctx, ctx->d_grp_rcv, ctx->grp_rcv.data(), ctx->grp_rcv.size() * 4);
  }
  std::vector<int32_t> idx((size_t)ctx->model.nslots, -1);
  for (size_t g = 0; g < ctx->grp_slot.size(); ++g) idx[ctx->grp_slot[g]] = (int32_t)g;
  upload_raw(ctx, ctx->d_pt_rcv, idx.data(), idx.size() * 4);
  ctx->data_valid = false;
}
}  // namespace dgrtm

extern "C" {

int rtm_set_receiver_capacity(dg_ctx* ctx, int64_t max_receivers) {
  DG_TRY(ctx)
  if (max_receivers < 0) throw ApiError(DG_ERR_ARG, "max_receivers must be >= 0");
  ctx->nr_reserve = max_receivers;
  DG_CATCH(ctx)
}

int rtm_image_device(dg_ctx* ctx, void** dptr, size_t* nbytes) {
  DG_TRY(ctx)
  require_history(ctx);
  if (!dptr || !nbytes) throw ApiError(DG_ERR_ARG, "dptr / nbytes is NULL");
  sync_stream(ctx);
  *dptr = ctx->image;
  *nbytes = (size_t)ctx->model.nblocks * ctx->Np * 32 * ctx->rs;
  DG_CATCH(ctx)
}

int rtm_spill_bytes(dg_ctx* ctx, int nsteps, size_t* n) {
  DG_TRY(ctx)
  if (!n) throw ApiError(DG_ERR_ARG, "n is NULL");
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  if (nsteps < 1) throw ApiError(DG_ERR_ARG, "nsteps must be >= 1");
  *n = spill_host_bytes(ctx, nsteps);
  DG_CATCH(ctx)
}

int rtm_set_trace_spill(dg_ctx* ctx, void* host, size_t n, int window) {
  DG_TRY(ctx)
  if (host && window < 2) throw ApiError(DG_ERR_ARG, "window must be >= 2 records");
  if (host && ((uintptr_t)host & 15) != 0) throw ApiError(DG_ERR_ARG, "host buffer must be 16-byte aligned");
  if (ctx->bound) sync_stream(ctx);
  if (ctx->copy_stream) cuda_check(cudaStreamSynchronize(ctx->copy_stream), "cudaStreamSynchronize (trace spill)");
  ctx->spill_host = (char*)host; ctx->spill_bytes = host ? n : 0; ctx->spill_window = host ? window : 0;
  ctx->hist_bound = false;                     // the record layout of the RTM region changed: bind it again
  DG_CATCH(ctx)
}

int rtm_set_spill_packing(dg_ctx* ctx, int on) {
  DG_TRY(ctx)
  if (on != 0 && on != 1) throw ApiError(DG_ERR_ARG, "on must be 0 or 1");
  if (ctx->bound) sync_stream(ctx);
  if (ctx->copy_stream) cuda_check(cudaStreamSynchronize(ctx->copy_stream), "cudaStreamSynchronize (trace spill)");
  ctx->spill_packed = on != 0;
  ctx->hist_bound = false;                     // host layout and the staging of the RTM region changed: bind it again
  DG_CATCH(ctx)
}

int rtm_history_bytes(dg_ctx* ctx, int nsteps, size_t* n) {
  DG_TRY(ctx)
  if (!n) throw ApiError(DG_ERR_ARG, "n is NULL");
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  if (nsteps < 1) throw ApiError(DG_ERR_ARG, "nsteps must be >= 1");
  HistPtrs keep;
  keep.save(ctx);
  Carver count;
  carve_history(ctx, count, nsteps);
  keep.restore(ctx);
  *n = count.used;
  DG_CATCH(ctx)
}

int rtm_bind_history(dg_ctx* ctx, void* dptr, size_t n) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!dptr || ((uintptr_t)dptr & 255) != 0) throw ApiError(DG_ERR_ARG, "device pointer must be non-NULL and 256-byte aligned");
  // the largest nsteps that fits decides the record capacity
  int nsteps = 0;
  {
    HistPtrs keep;
    keep.save(ctx);
    int lo = 0, hi = 1;
    auto fits = [&](int s) {
      Carver cnt; carve_history(ctx, cnt, s);
      return cnt.used <= n && (ctx->spill_window <= 0 || spill_host_bytes(ctx, s) <= ctx->spill_bytes);
    };
    if (fits(1)) {
      lo = 1;
      while (hi < (1 << 28) && fits(hi * 2)) hi *= 2;
      lo = hi; hi = hi * 2;
      while (hi - lo > 1) { const int mid = lo + (hi - lo) / 2; if (fits(mid)) lo = mid; else hi = mid; }
    }
    keep.restore(ctx);
    nsteps = lo;
  }
  if (nsteps < 1) throw ApiError(DG_ERR_NOMEM, "history buffer too small for a single step");
  ctx->hs = (char*)dptr; ctx->hs_bytes = n; ctx->hist_nsteps = nsteps;
  Carver cv;
  cv.base = ctx->hs;
  carve_history(ctx, cv, nsteps);
  spill_setup(ctx, nsteps);
  ctx->nr_cap = std::max(ctx->nr, ctx->nr_reserve);
  upload_receiver_tables(ctx);
  ctx->hist_bound = true;
  clear_field(ctx, ctx->R);
  cuda_check(cudaMemsetAsync(ctx->image, 0, (size_t)ctx->model.nblocks * ctx->Np * 32 * ctx->rs, ctx->stream), "memset image");
  ctx->have_final = false; ctx->have_backward = false;
  sync_stream(ctx);
  DG_CATCH(ctx)
}

// A phase of a shot in parts (rtm_forward_part / rtm_backward_part, include/dgrtm.h): fine steps [fine0, fine0 + nfine) of
// the phase; the part that starts at 0 initialises the phase, the part that reaches its end finishes it.
static void forward_part(dg_ctx* ctx, int nsteps, int64_t fine0, int64_t nfine, double* data_out) {
  require_history(ctx);
  if (nsteps < 1 || nsteps > ctx->hist_nsteps) throw ApiError(DG_ERR_NOMEM, "nsteps exceeds the bound history capacity (" + std::to_string(ctx->hist_nsteps) + ")");
  if (ctx->integrator != DG_INTEGRATOR_AB3) throw ApiError(DG_ERR_UNSUPPORTED, "RTM uses the AB3 / multi-rate AB3 integrator");
  const int64_t total = (int64_t)nsteps * ctx->nlocal;
  if (fine0 < 0 || nfine < 0 || fine0 + nfine > total) throw ApiError(DG_ERR_ARG, "fine steps outside the forward phase");
  if (fine0 == 0 && !(ctx->part_phase == 1 && ctx->part_nsteps == nsteps && ctx->part_fresh)) {   // (an empty first part
    clear_field(ctx, ctx->F);                                // initialises alone, so that the trace buffers can be asked for)
    ctx->t0 = 0; ctx->fine = 0;
    ctx->have_final = false; ctx->have_backward = false;
    ctx->part_phase = 1; ctx->part_nsteps = nsteps; ctx->part_fresh = true;
  } else if (ctx->part_phase != 1 || ctx->part_nsteps != nsteps || ctx->fine != fine0) {
    throw ApiError(DG_ERR_STATE, "the parts of a forward phase follow one another from fine step 0");
  }
  RunOpts o;
  o.direction = 1; o.fields[0] = &ctx->F; o.nfields = 1; o.source_on[0] = ctx->has_src;
  o.capture = true; o.record = ctx->nr > 0;
  o.first_fine = fine0; o.t0 = (double)fine0 * ctx->dt_local;
  o.fine_phase = fine0 % ctx->nlocal; o.nfine = nfine; o.finish = fine0 + nfine == total;
  run_mrab(ctx, 0, o);
  ctx->fine = fine0 + nfine;
  if (nfine > 0) ctx->part_fresh = false;
  if (o.finish) {
    cuda_check(cudaMemcpyAsync(ctx->qfinal, ctx->F.q, field_bytes(ctx), cudaMemcpyDeviceToDevice, ctx->stream), "save final state");
    ctx->have_final = true; ctx->final_nsteps = nsteps;
    ctx->data_valid = ctx->nr > 0;
    ctx->part_phase = 0;
  }
  check_launches(ctx);
  if (o.finish) {
    if (data_out) copy_data(ctx, data_out, nullptr, total + 1);
    sync_stream(ctx);
    if (ctx->spill_window > 0) cuda_check(cudaStreamSynchronize(ctx->copy_stream), "cudaStreamSynchronize (trace spill)");
  }
}

static void backward_part(dg_ctx* ctx, int nsteps, const double* data, const double updir[3], int imaging,
                          int64_t first_image_step, int64_t fine0, int64_t nfine) {
  require_history(ctx);
  if (!ctx->have_final) throw ApiError(DG_ERR_STATE, "rtm_forward_shot first");
  if (nsteps < 1 || nsteps > ctx->final_nsteps) throw ApiError(DG_ERR_ARG, "nsteps must be in 1..(steps of the forward shot)");
  if (!updir) throw ApiError(DG_ERR_ARG, "updir is NULL");
  if (imaging < 0 || imaging > 3) throw ApiError(DG_ERR_ARG, "unknown imaging condition");
  const int64_t ntot = ctx->final_nsteps, total = (int64_t)nsteps * ctx->nlocal;
  if (fine0 < 0 || nfine < 0 || fine0 + nfine > total) throw ApiError(DG_ERR_ARG, "fine steps outside the backward phase");
  if (fine0 == 0 && (data || !(ctx->part_phase == 2 && ctx->part_nsteps == nsteps && ctx->part_fresh))) {   // (signals given: a new start)
    if (!data && ctx->nr > 0 && !ctx->data_valid)
      throw ApiError(DG_ERR_STATE, "the signals on the device belong to another receiver set: pass data");
    if (data) ctx->data_valid = true;
    if (data) copy_data(ctx, nullptr, data, ntot * ctx->nlocal + 1);   // NULL: the signals recorded on the device
    // source field: restart from q(t_f) (history restarts, reading Q7); receiver field: from rest
    cuda_check(cudaMemcpyAsync(ctx->F.q, ctx->qfinal, field_bytes(ctx), cudaMemcpyDeviceToDevice, ctx->stream), "restore final state");
    for (int s = 0; s < 3; ++s) cuda_check(cudaMemsetAsync(ctx->F.hist[s], 0, field_bytes(ctx), ctx->stream), "memset hist");
    ctx->F.reset_history();
    refresh_traces(ctx, ctx->F);
    clear_field(ctx, ctx->R);
    ctx->part_phase = 2; ctx->part_nsteps = nsteps; ctx->part_fresh = true;
    ctx->fine = ntot * ctx->nlocal;
  } else if (ctx->part_phase != 2 || ctx->part_nsteps != nsteps || ctx->fine != ntot * ctx->nlocal - fine0) {
    throw ApiError(DG_ERR_STATE, "the parts of a backward phase follow one another from fine step 0");
  }
  RunOpts o;
  o.direction = -1; o.fields[0] = &ctx->F; o.fields[1] = &ctx->R; o.nfields = 2;
  o.source_on[0] = ctx->has_src; o.source_on[1] = false;
  o.replay = true; o.inject_field = ctx->nr > 0 ? 1 : -1;
  o.image = true; o.imaging = imaging;
  for (int d = 0; d < 3; ++d) o.updir[d] = updir[d];
  o.image_min_fine = first_image_step * ctx->nlocal;
  o.first_fine = ntot * ctx->nlocal - fine0;
  o.t0 = (double)o.first_fine * ctx->dt_local;
  o.fine_phase = fine0 % ctx->nlocal; o.nfine = nfine; o.finish = fine0 + nfine == total;
  run_mrab(ctx, 0, o);
  ctx->fine = o.first_fine - nfine;
  if (nfine > 0) ctx->part_fresh = false;
  check_launches(ctx);
  if (o.finish) { ctx->have_backward = true; ctx->part_phase = 0; sync_stream(ctx); }
}

int rtm_forward_shot(dg_ctx* ctx, int nsteps, double* data_out) {
  DG_TRY(ctx)
  forward_part(ctx, nsteps, 0, (int64_t)nsteps * ctx->nlocal, data_out);
  DG_CATCH(ctx)
}

int rtm_backward_shot(dg_ctx* ctx, int nsteps, const double* data, const double updir[3], int imaging,
                      int64_t first_image_step) {
  DG_TRY(ctx)
  backward_part(ctx, nsteps, data, updir, imaging, first_image_step, 0, (int64_t)nsteps * ctx->nlocal);
  DG_CATCH(ctx)
}

int rtm_forward_part(dg_ctx* ctx, int nsteps, int64_t fine0, int64_t nfine, double* data_out) {
  DG_TRY(ctx)
  forward_part(ctx, nsteps, fine0, nfine, data_out);
  DG_CATCH(ctx)
}

int rtm_backward_part(dg_ctx* ctx, int nsteps, const double* data, const double updir[3], int imaging,
                      int64_t first_image_step, int64_t fine0, int64_t nfine) {
  DG_TRY(ctx)
  backward_part(ctx, nsteps, data, updir, imaging, first_image_step, fine0, nfine);
  DG_CATCH(ctx)
}

int rtm_get_trace_levels(dg_ctx* ctx, int field, void** current, void** half, size_t* nbytes) {
  DG_TRY(ctx)
  require_history(ctx);
  if (field != 0 && field != 1) throw ApiError(DG_ERR_ARG, "field must be 0 (source) or 1 (receivers)");
  if (!current || !half || !nbytes) throw ApiError(DG_ERR_ARG, "current / half / nbytes is NULL");
  Field& F = field == 0 ? ctx->F : ctx->R;
  for (int l = 0; l < ctx->model.nlevels; ++l) current[l] = F.qfb[F.par[l]];
  *half = F.qfh;
  *nbytes = trace_bytes(ctx);
  DG_CATCH(ctx)
}

int dg_get_trace_buffers(dg_ctx* ctx, int field, void** buffers, size_t* nbytes) {
  DG_TRY(ctx)
  if (field == 0) require_bound(ctx); else require_history(ctx);
  if (field != 0 && field != 1) throw ApiError(DG_ERR_ARG, "field must be 0 (source) or 1 (receivers)");
  if (!buffers || !nbytes) throw ApiError(DG_ERR_ARG, "buffers / nbytes is NULL");
  Field& F = field == 0 ? ctx->F : ctx->R;
  buffers[0] = F.qfb[0]; buffers[1] = F.qfb[1]; buffers[2] = F.qfh;
  *nbytes = trace_bytes(ctx);
  DG_CATCH(ctx)
}

int rtm_halo_sources(dg_ctx* ctx, int nsets, const void* const* src_trace_device) {
  DG_TRY(ctx)
  require_history(ctx);
  if (nsets < 0 || nsets > kMaxHaloSets) throw ApiError(DG_ERR_ARG, "nsets must be in 0..32");
  if (nsets && !src_trace_device) throw ApiError(DG_ERR_ARG, "source table is NULL");
  for (int x = 0; x < kMaxHaloSets; ++x) {
    const void* p = x < nsets ? src_trace_device[x] : nullptr;
    if (!p && ctx->halo_off[x + 1] > ctx->halo_off[x]) throw ApiError(DG_ERR_ARG, "a non-empty halo set has no source");
    ctx->halo_src2[x] = p;
  }
  ctx->halo_src2_valid = true;
  DG_CATCH(ctx)
}

int rtm_image_read(dg_ctx* ctx, double* I_out) {
  DG_TRY(ctx)
  require_history(ctx);
  if (!I_out) throw ApiError(DG_ERR_ARG, "I_out is NULL");
  image_from_device(ctx, I_out, ctx->image);
  DG_CATCH(ctx)
}

int rtm_image_zero(dg_ctx* ctx) {
  DG_TRY(ctx)
  require_history(ctx);
  cuda_check(cudaMemsetAsync(ctx->image, 0, (size_t)ctx->model.nblocks * ctx->Np * 32 * ctx->rs, ctx->stream), "memset image");
  DG_CATCH(ctx)
}

int rtm_get_trace_index(const dg_ctx* ctx, int level, int64_t* nfaces, int64_t* nrecords, int32_t* faces) {
  if (!ctx) return DG_ERR_ARG;
  if (!ctx->has_model || level < 0 || level >= ctx->model.nlevels) return DG_ERR_ARG;
  const std::vector<int32_t>& st = ctx->model.stored[level];
  if (nfaces) *nfaces = (int64_t)st.size();
  if (nrecords) *nrecords = ctx->hist_bound ? records_of_level(ctx, level, ctx->have_final ? ctx->final_nsteps : ctx->hist_nsteps) : 0;
  if (faces) std::copy(st.begin(), st.end(), faces);
  return DG_OK;
}

int rtm_get_traces(dg_ctx* ctx, int level, int64_t record, double* buf) {
  DG_TRY(ctx)
  require_history(ctx);
  if (!buf || level < 0 || level >= ctx->model.nlevels) throw ApiError(DG_ERR_ARG, "bad level / buffer");
  if (record < 0 || record >= records_of_level(ctx, level, ctx->hist_nsteps)) throw ApiError(DG_ERR_ARG, "record out of range");
  const size_t nf = ctx->model.stored[level].size(), Nfp = ctx->Nfp;
  std::vector<double> tmp(nf * 2 * Nfp);
  if (ctx->spill_window > 0) {                 // the host copy is the history
    sync_stream(ctx);
    cuda_check(cudaStreamSynchronize(ctx->copy_stream), "cudaStreamSynchronize (trace spill)");
    if (ctx->spill_packed) {                   // fp32 / bf16 values of the packed host copy
      const char* src = ctx->hrec[level] + (size_t)record * nf * ctx->REC * (ctx->rs / 2);
      for (size_t i = 0; i < tmp.size(); ++i) {
        if (ctx->precision == 64) tmp[i] = (double)((const float*)src)[i];
        else { const uint32_t bits = (uint32_t)((const uint16_t*)src)[i] << 16; float f; std::memcpy(&f, &bits, 4); tmp[i] = (double)f; }
      }
    } else {
      const char* src = ctx->hrec[level] + (size_t)record * nf * ctx->REC * ctx->rs;
      for (size_t i = 0; i < tmp.size(); ++i) tmp[i] = ctx->precision == 64 ? ((const double*)src)[i] : (double)((const float*)src)[i];
    }
  } else {
    download_real(ctx, tmp.data(), ctx->rec[level] + (size_t)record * nf * ctx->REC * ctx->rs, tmp.size());
  }
  // device record: [face][p | n.v][Nfp]  ->  buf[face][Nfp][2]
  for (size_t x = 0; x < nf; ++x)
    for (size_t i = 0; i < Nfp; ++i) {
      buf[(x * Nfp + i) * 2 + 0] = tmp[x * 2 * Nfp + i];
      buf[(x * Nfp + i) * 2 + 1] = tmp[x * 2 * Nfp + Nfp + i];
    }
  DG_CATCH(ctx)
}

int rtm_get_fields(dg_ctx* ctx, int which, double* q) {
  DG_TRY(ctx)
  require_history(ctx);
  if (!q) throw ApiError(DG_ERR_ARG, "q is NULL");
  if (which == 0) {
    if (!ctx->have_final) throw ApiError(DG_ERR_STATE, "rtm_forward_shot first");
    fields_from_device(ctx, q, ctx->qfinal);
  } else if (which == 1 || which == 2) {
    if (!ctx->have_backward) throw ApiError(DG_ERR_STATE, "rtm_backward_shot first");
    fields_from_device(ctx, q, which == 1 ? ctx->F.q : ctx->R.q);
  } else {
    throw ApiError(DG_ERR_ARG, "which must be 0, 1 or 2");
  }
  DG_CATCH(ctx)
}

}  // extern "C"
