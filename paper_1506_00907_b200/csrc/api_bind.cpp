// C ABI of libdgrtm, part 2: binding caller-owned device memory, uploading the tables of the
// level-sorted, 32-element-blocked layout (kernels.h), initial state.
#include <algorithm>

#include "ctx.h"

using namespace dgrtm;

namespace dgrtm {
void upload_point_source(dg_ctx* c) {
  std::vector<int32_t> idx((size_t)c->model.nslots, -1);
  if (c->has_src) idx[c->model.slot_of[c->src_k]] = 0;
  upload_raw(c, c->d_pt_src, idx.data(), idx.size() * 4);
}
}  // namespace dgrtm

namespace {

void upload_tables(dg_ctx* c) {
  const int Np = c->Np, Nfp = c->Nfp, NF = c->NF;
  const RefElem& re = c->re;
  const Mesh& m = c->mesh;
  const Model& md = c->model;
  // operators, transposed for the kernels: D3T[m][n][3] = D_{r,s,t}[n][m]; LIFTT[j][n] = LIFT[n][j]
  std::vector<double> D3T((size_t)3 * Np * Np), LT((size_t)NF * Np);
  for (int mm = 0; mm < Np; ++mm)
    for (int n = 0; n < Np; ++n) {
      D3T[((size_t)mm * Np + n) * 3 + 0] = re.Dr[(size_t)n * Np + mm];
      D3T[((size_t)mm * Np + n) * 3 + 1] = re.Ds[(size_t)n * Np + mm];
      D3T[((size_t)mm * Np + n) * 3 + 2] = re.Dt[(size_t)n * Np + mm];
    }
  for (int j = 0; j < NF; ++j)
    for (int n = 0; n < Np; ++n) LT[(size_t)j * Np + n] = re.LIFT[(size_t)n * NF + j];
  upload_real(c, const_cast<void*>(c->ops.D3T), D3T.data(), D3T.size());
  upload_real(c, const_cast<void*>(c->ops.LIFTT), LT.data(), LT.size());
  {  // step kernel: D3P[m][3][NPAD] = D_{r,s,t}[n][m], LTP[j][NPAD] = LIFT[n][j], zero-padded in n
    const int npad = c->kt->step_npad;
    std::vector<double> D3P((size_t)3 * Np * npad, 0.0), LTP((size_t)NF * npad, 0.0);
    for (int mm = 0; mm < Np; ++mm)
      for (int n = 0; n < Np; ++n) {
        D3P[((size_t)mm * 3 + 0) * npad + n] = re.Dr[(size_t)n * Np + mm];
        D3P[((size_t)mm * 3 + 1) * npad + n] = re.Ds[(size_t)n * Np + mm];
        D3P[((size_t)mm * 3 + 2) * npad + n] = re.Dt[(size_t)n * Np + mm];
      }
    for (int j = 0; j < NF; ++j)
      for (int n = 0; n < Np; ++n) LTP[(size_t)j * npad + n] = re.LIFT[(size_t)n * NF + j];
    upload_real(c, c->d_D3P, D3P.data(), D3P.size());
    upload_real(c, c->d_LTP, LTP.data(), LTP.size());
    if (c->kt->pipe) {   // tile-packed: D3Q[w][m][RL] = (Dr, Ds, Dt)[n0 + nn][m], LTQ[w][j][LL] = LIFT[n0 + nn][j]
      const int TO = c->kt->pipe_TO, NT = c->kt->pipe_NT, RL = c->kt->pipe_RL, LL = c->kt->pipe_LL;
      std::vector<double> D3Q((size_t)NT * Np * RL, 0.0), LTQ((size_t)NT * NF * LL, 0.0);
      for (int w = 0; w < NT; ++w)
        for (int nn = 0; nn < TO; ++nn) {
          const int n = w * TO + nn;
          if (n >= Np) continue;
          for (int mm = 0; mm < Np; ++mm) {
            double* row = &D3Q[((size_t)w * Np + mm) * RL];
            row[nn] = re.Dr[(size_t)n * Np + mm]; row[TO + nn] = re.Ds[(size_t)n * Np + mm]; row[2 * TO + nn] = re.Dt[(size_t)n * Np + mm];
          }
          for (int j = 0; j < NF; ++j) LTQ[((size_t)w * NF + j) * LL + nn] = re.LIFT[(size_t)n * NF + j];
        }
      // the kernel's table image: reals (device precision) then Fmask and the permutation table
      std::vector<char> blob(c->kt->pipe_blob_bytes, 0);
      size_t off = 0;
      auto put_reals = [&](const std::vector<double>& v) {
        for (double x : v) {
          if (c->precision == 64) { std::memcpy(&blob[off], &x, 8); off += 8; }
          else { const float f = (float)x; std::memcpy(&blob[off], &f, 4); off += 4; }
        }
      };
      put_reals(D3Q); put_reals(LTQ);
      std::memcpy(&blob[off], re.Fmask.data(), (size_t)NF * 4); off += (size_t)NF * 4;
      if (off + m.ptab.size() * 4 > blob.size()) throw ApiError(DG_ERR_UNSUPPORTED, "too many distinct face permutations");
      std::memcpy(&blob[off], m.ptab.data(), m.ptab.size() * 4);
      upload_raw(c, c->d_D3Q, blob.data(), blob.size());
    }
    if (c->kt->tc) {     // tensor-core kernel: B tables in the canonical K-major no-swizzle layout, split hi / lo (TF32)
      const int K1 = c->kt->tc_K1, K2 = c->kt->tc_K2, NN = c->kt->tc_NN;
      auto tf32 = [](float x) {             // round to nearest even at 10 mantissa bits
        uint32_t u; std::memcpy(&u, &x, 4);
        u = (u + 0x0FFFu + ((u >> 13) & 1u)) & 0xFFFFE000u;
        float y; std::memcpy(&y, &u, 4); return y;
      };
      auto idx = [NN](int kap, int n) { return (size_t)(kap / 8) * (8 * NN) + ((size_t)(((kap % 8) / 4) * NN + n) * 4 + (kap % 4)); };
      std::vector<float> B1h((size_t)K1 * NN, 0.f), B1l(B1h), B2h((size_t)K2 * NN, 0.f), B2l(B2h);
      for (int j = 0; j < 3; ++j)
        for (int mm = 0; mm < Np; ++mm)
          for (int n = 0; n < Np; ++n) {
            const std::vector<double>& D = j == 0 ? re.Dr : (j == 1 ? re.Ds : re.Dt);
            const double v = D[(size_t)n * Np + mm];
            const float h = tf32((float)v);
            B1h[idx(j * Np + mm, n)] = h; B1l[idx(j * Np + mm, n)] = tf32((float)(v - (double)h));
          }
      for (int j = 0; j < NF; ++j)
        for (int n = 0; n < Np; ++n) {
          const double v = re.LIFT[(size_t)n * NF + j];
          const float h = tf32((float)v);
          B2h[idx(j, n)] = h; B2l[idx(j, n)] = tf32((float)(v - (double)h));
        }
      std::vector<char> blob(c->kt->tc_blob_bytes, 0);
      size_t off = 0;
      for (const std::vector<float>* t : {&B1h, &B1l, &B2h, &B2l}) { std::memcpy(&blob[off], t->data(), t->size() * 4); off += t->size() * 4; }
      std::memcpy(&blob[off], re.Fmask.data(), (size_t)NF * 4); off += (size_t)NF * 4;
      if (off + m.ptab.size() * 4 > blob.size()) throw ApiError(DG_ERR_UNSUPPORTED, "too many distinct face permutations");
      std::memcpy(&blob[off], m.ptab.data(), m.ptab.size() * 4);
      upload_raw(c, c->d_LTQ, blob.data(), blob.size());
    }
  }
  upload_raw(c, const_cast<int*>(c->ops.Fmask), re.Fmask.data(), (size_t)NF * 4);
  upload_raw(c, const_cast<int*>(c->ops.ptab), m.ptab.data(), m.ptab.size() * 4);

  // position of every stored (absorbing) boundary face inside its level's record
  std::vector<int32_t> stored_pos(m.bnd_k.size(), 0);
  for (int l = 0; l < md.nlevels; ++l)
    for (size_t x = 0; x < md.stored[l].size(); ++x) stored_pos[md.stored[l][x]] = (int32_t)x;

  const int64_t nb = md.nblocks;
  std::vector<double> geo((size_t)nb * DG_NGEO * 32, 0.0);
  std::vector<int32_t> nbr((size_t)nb * 4 * 32, -1), wperm((size_t)nb * 32, 0);
  for (int64_t s = 0; s < md.nslots; ++s) {
    const int64_t k = md.elem_of[s], b = s >> 5, lane = s & 31;
    double* g = &geo[(size_t)b * DG_NGEO * 32 + lane];
    if (k < 0) {                                   // padding slot: inert
      for (int f = 0; f < 4; ++f) g[(GEO_FACE + 5 * f + 4) * 32] = 1.0;
      g[GEO_IRHO * 32] = 1.0;
      continue;
    }
    const double rho = md.rho[k], cc = md.c[k], Z = rho * cc;
    for (int x = 0; x < 9; ++x) g[(GEO_G + x) * 32] = m.ginv[9 * k + x];
    g[GEO_RC2 * 32] = rho * cc * cc;
    g[GEO_IRHO * 32] = 1.0 / rho;
    g[GEO_Z * 32] = Z;
    int wp = 0;
    for (int f = 0; f < 4; ++f) {
      const int64_t k2 = m.EToE[4 * k + f];
      for (int d = 0; d < 3; ++d) g[(GEO_FACE + 5 * f + d) * 32] = m.normals[12 * k + 3 * f + d];
      g[(GEO_FACE + 5 * f + 3) * 32] = m.gsur[4 * k + f];
      // single-valued face impedance (reading Q4)
      g[(GEO_FACE + 5 * f + 4) * 32] = k2 >= 0 ? 0.5 * (Z + md.rho[k2] * md.c[k2]) : Z;
      if (k2 < 0 && !c->bnd_Zext.empty()) {        // halo face: the neighbouring sub-domain's impedance (dg_set_exterior_impedance)
        const double Ze = c->bnd_Zext[m.bnd_index[4 * k + f]];
        if (Ze > 0) g[(GEO_FACE + 5 * f + 4) * 32] = 0.5 * (Z + Ze);
      }
      int32_t code;
      if (k2 >= 0) {
        code = (int32_t)(md.slot_of[k2] * 4 + m.EToF[4 * k + f]);
      } else {
        const int bc = m.bc[4 * k + f];
        const int32_t bi = m.bnd_index[4 * k + f];
        const int64_t bpos = bc == DG_BC_ABSORBING ? stored_pos[bi] : (bc == DG_BC_PRESCRIBED ? bi : 0);
        code = (int32_t)(-1 - (bpos * 8 + bc));
      }
      nbr[((size_t)b * 4 + f) * 32 + lane] = code;
      wp |= (int)m.perm_id[4 * k + f] << (8 * f);
    }
    wperm[s] = wp;
  }
  upload_real(c, c->geo, geo.data(), geo.size());
  upload_raw(c, c->nbr, nbr.data(), nbr.size() * 4);
  upload_raw(c, c->wperm, wperm.data(), wperm.size() * 4);

  for (int l = 0; l < md.nlevels; ++l) {
    std::vector<int32_t> sf(md.stored[l].size());
    for (size_t x = 0; x < sf.size(); ++x) {
      const int32_t bi = md.stored[l][x];
      sf[x] = (int32_t)(md.slot_of[m.bnd_k[bi]] * 4 + m.bnd_f[bi]);
    }
    upload_raw(c, c->d_stored[l], sf.data(), sf.size() * 4);
  }
  if (c->has_src) upload_real(c, c->d_src_w, c->src_w.data(), Np);
  std::vector<unsigned char> flag((size_t)md.nblocks + 32, 0);   // block flags, then the zeroed ticket counters
  for (int l = 0; l < md.nlevels; ++l)
    for (int32_t s : md.coarse_nb[l]) flag[s >> 5] |= 1;
  upload_raw(c, c->d_blkflag, flag.data(), flag.size());
  c->sched_sel = 0;
  upload_point_source(c);
}

}  // namespace

extern "C" {

int dg_bind_workspace(dg_ctx* ctx, void* dptr, size_t n, void* cuda_stream) {
  DG_TRY(ctx)
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  if (!dptr) throw ApiError(DG_ERR_ARG, "device pointer is NULL");
  if (((uintptr_t)dptr & 255) != 0) throw ApiError(DG_ERR_ARG, "device pointer must be 256-byte aligned");
  size_t need = 0;
  int rc = dg_workspace_bytes(ctx, &need);
  if (rc != DG_OK) return rc;
  if (n < need) throw ApiError(DG_ERR_NOMEM, "workspace too small: need " + std::to_string(need) + " bytes");
  if (!ctx->kt) throw ApiError(DG_ERR_UNSUPPORTED, "no kernels for this order / precision");
  const int e = ctx->kt->init();
  if (e != 0) throw ApiError(DG_ERR_CUDA, std::string("kernel attribute setup: ") + cudaGetErrorString((cudaError_t)e));
  ctx->ws = (char*)dptr; ctx->ws_bytes = n; ctx->stream = (cudaStream_t)cuda_stream;
  Carver cv;
  cv.base = ctx->ws;
  carve_workspace(ctx, cv);
  ctx->bound = true; ctx->hist_bound = false;
  cuda_check(cudaMemsetAsync(ctx->ws, 0, need, ctx->stream), "cudaMemsetAsync workspace");
  upload_tables(ctx);
  ctx->F.reset_history();
  ctx->t0 = 0; ctx->fine = 0; ctx->has_ext = false; for (int x = 0; x <= kMaxHaloSets; ++x) ctx->halo_off[x] = 0;
  {
    const size_t nbf = ctx->mesh.bnd_k.size();
    ctx->h_hrec.assign(nbf, -1); ctx->h_hset.assign(nbf, 0); ctx->h_hpos.assign(nbf * ctx->Nfp, 0);
    if (nbf) upload_raw(ctx, ctx->d_halo_face, ctx->h_hrec.data(), nbf * 8);   // -1: no face is a halo face yet
    ctx->halo_src_valid = false; ctx->halo_src2_valid = false;
  }
  ctx->have_final = false; ctx->have_backward = false;
  sync_stream(ctx);
  DG_CATCH(ctx)
}

int dg_set_state(dg_ctx* ctx, const double* q, double t0) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!q) throw ApiError(DG_ERR_ARG, "q is NULL");
  clear_field(ctx, ctx->F);
  cuda_check(cudaMemsetAsync(ctx->scratch, 0, field_bytes(ctx), ctx->stream), "memset scratch");
  fields_to_device(ctx, ctx->F.q, q);
  refresh_traces(ctx, ctx->F);
  ctx->t0 = t0; ctx->fine = 0;
  sync_stream(ctx);
  DG_CATCH(ctx)
}

// ---- domain decomposition: halo faces -----------------------------
int dg_set_exterior_impedance(dg_ctx* ctx, const double* Zext) {
  DG_TRY(ctx)
  const size_t nb = ctx->mesh.bnd_k.size();
  if (Zext) ctx->bnd_Zext.assign(Zext, Zext + nb); else ctx->bnd_Zext.clear();
  ctx->bound = false; ctx->hist_bound = false;   // the face impedances live in the bound factors: bind again
  DG_CATCH(ctx)
}

int dg_get_slots(dg_ctx* ctx, int64_t* slot_of) {
  DG_TRY(ctx)
  if (!slot_of) throw ApiError(DG_ERR_ARG, "slot_of is NULL");
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  for (int64_t k = 0; k < ctx->mesh.K; ++k) slot_of[k] = ctx->model.slot_of[k];
  DG_CATCH(ctx)
}

int dg_get_trace_device(dg_ctx* ctx, void** dptr, size_t* nbytes) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!dptr || !nbytes) throw ApiError(DG_ERR_ARG, "dptr / nbytes is NULL");
  if (ctx->model.nlevels != 1) throw ApiError(DG_ERR_UNSUPPORTED, "the halo exchange is single-rate");
  *dptr = ctx->F.qfb[ctx->F.par[0]];
  *nbytes = trace_bytes(ctx);
  DG_CATCH(ctx)
}

int dg_get_trace_levels(dg_ctx* ctx, void** current, void** half, size_t* nbytes) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!current || !half || !nbytes) throw ApiError(DG_ERR_ARG, "current / half / nbytes is NULL");
  for (int l = 0; l < ctx->model.nlevels; ++l) current[l] = ctx->F.qfb[ctx->F.par[l]];
  *half = ctx->F.qfh;
  *nbytes = trace_bytes(ctx);
  DG_CATCH(ctx)
}

int dg_set_halo(dg_ctx* ctx, int set, int64_t nh, const int32_t* bnd_index, const int64_t* src_record, const int32_t* src_pos) {
  DG_TRY(ctx)
  require_bound(ctx);
  const int64_t nb = (int64_t)ctx->mesh.bnd_k.size();
  const int Nfp = ctx->Nfp;
  if (set < 0 || set >= kMaxHaloSets) throw ApiError(DG_ERR_ARG, "halo set must be in 0..31");
  const int64_t h0 = ctx->halo_off[set];          // sets are filled in ascending order: set s starts where s - 1 ended
  if (nh < 0 || h0 + nh > nb) throw ApiError(DG_ERR_ARG, "more halo faces than boundary faces");
  if (nh && (!bnd_index || !src_record || !src_pos)) throw ApiError(DG_ERR_ARG, "NULL table");
  for (int64_t h = 0; h < nh; ++h) {
    const int32_t bi = bnd_index[h];
    if (bi < 0 || bi >= nb) throw ApiError(DG_ERR_ARG, "boundary-face index out of range");
    if (ctx->mesh.bc[4 * (size_t)ctx->mesh.bnd_k[bi] + ctx->mesh.bnd_f[bi]] != DG_BC_PRESCRIBED)
      throw ApiError(DG_ERR_ARG, "halo faces must be DG_BC_PRESCRIBED faces");
    if (src_record[h] < 0) throw ApiError(DG_ERR_ARG, "negative source record");
    for (int i = 0; i < Nfp; ++i)
      if (src_pos[h * Nfp + i] < 0 || src_pos[h * Nfp + i] >= Nfp) throw ApiError(DG_ERR_ARG, "source node position out of range");
  }
  // carved region: [bnd int32 nb | pad to 8 | rec int64 nb | pos int32 nb*Nfp], the sets one after the other
  char* base = ctx->d_halo;
  const size_t off_rec = ((size_t)nb * 4 + 7) / 8 * 8, off_pos = off_rec + (size_t)nb * 8;
  if (nh) {
    upload_raw(ctx, base + (size_t)h0 * 4, bnd_index, (size_t)nh * 4);
    upload_raw(ctx, base + off_rec + (size_t)h0 * 8, src_record, (size_t)nh * 8);
    upload_raw(ctx, base + off_pos + (size_t)h0 * Nfp * 4, src_pos, (size_t)nh * Nfp * 4);
  }
  if (!ctx->has_ext) {   // prescribed faces that are no halo faces keep a zero exterior until dg_set_exterior
    cuda_check(cudaMemsetAsync(ctx->ext, 0, std::max<size_t>(1, (size_t)nb) * Nfp * 2 * ctx->rs, ctx->stream), "memset ext");
    ctx->has_ext = true;
  }
  for (int x = set + 1; x <= kMaxHaloSets; ++x) ctx->halo_off[x] = h0 + nh;
  // the same tables by boundary face (fused exchange, dg_halo_sources): [hrec int64 nb | hset int32 nb | hpos int32 nb*Nfp]
  for (int64_t h = 0; h < nh; ++h) {
    const size_t bi = (size_t)bnd_index[h];
    ctx->h_hrec[bi] = src_record[h]; ctx->h_hset[bi] = set;
    for (int i = 0; i < Nfp; ++i) ctx->h_hpos[bi * Nfp + i] = src_pos[h * Nfp + i];
  }
  if (nb) {
    upload_raw(ctx, ctx->d_halo_face, ctx->h_hrec.data(), (size_t)nb * 8);
    upload_raw(ctx, ctx->d_halo_face + (size_t)nb * 8, ctx->h_hset.data(), (size_t)nb * 4);
    upload_raw(ctx, ctx->d_halo_face + (size_t)nb * 12, ctx->h_hpos.data(), (size_t)nb * Nfp * 4);
  }
  DG_CATCH(ctx)
}

int dg_halo_sources(dg_ctx* ctx, int nsets, const void* const* src_trace_device) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (nsets < 0 || nsets > kMaxHaloSets) throw ApiError(DG_ERR_ARG, "nsets must be in 0..32");
  if (nsets && !src_trace_device) throw ApiError(DG_ERR_ARG, "source table is NULL");
  if (ctx->integrator != DG_INTEGRATOR_AB3 || ctx->use_tc)
    throw ApiError(DG_ERR_UNSUPPORTED, "the fused halo exchange is in the AB step kernels (k_pipe, k_step): use dg_halo_pull");
  for (int x = 0; x < nsets; ++x) {
    if (!src_trace_device[x] && ctx->halo_off[x + 1] > ctx->halo_off[x]) throw ApiError(DG_ERR_ARG, "NULL source of a non-empty halo set");
    ctx->halo_src[x] = src_trace_device[x];
  }
  for (int x = nsets; x < kMaxHaloSets; ++x) {
    if (ctx->halo_off[x + 1] > ctx->halo_off[x]) throw ApiError(DG_ERR_ARG, "a non-empty halo set has no source");
    ctx->halo_src[x] = nullptr;
  }
  ctx->halo_src_valid = true;
  DG_CATCH(ctx)
}

int dg_halo_pull(dg_ctx* ctx, int set, const void* src_trace_device) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (set < 0 || set >= kMaxHaloSets) throw ApiError(DG_ERR_ARG, "halo set must be in 0..31");
  if (!src_trace_device) throw ApiError(DG_ERR_ARG, "source trace buffer is NULL");
  const int64_t h0 = ctx->halo_off[set], nh = ctx->halo_off[set + 1] - h0;
  if (nh > 0) {
    const size_t nb = ctx->mesh.bnd_k.size();
    const size_t off_rec = (nb * 4 + 7) / 8 * 8, off_pos = off_rec + nb * 8;
    HaloArgs a;
    a.src_qf = src_trace_device; a.ext = ctx->ext;
    a.bnd = reinterpret_cast<const int*>(ctx->d_halo) + h0;
    a.rec = reinterpret_cast<const long long*>(ctx->d_halo + off_rec) + h0;
    a.pos = reinterpret_cast<const int*>(ctx->d_halo + off_pos) + (size_t)h0 * ctx->Nfp;
    a.nh = (int)nh;
    DG_LAUNCH(ctx, KC_HALO, ctx->kt->halo(a, ctx->stream));
    check_launches(ctx);
  }
  DG_CATCH(ctx)
}

int dg_set_exterior(dg_ctx* ctx, const double* ext) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!ext) throw ApiError(DG_ERR_ARG, "ext is NULL");
  upload_real(ctx, ctx->ext, ext, ctx->mesh.bnd_k.size() * ctx->Nfp * 2);
  ctx->has_ext = true;
  DG_CATCH(ctx)
}

}  // extern "C"
