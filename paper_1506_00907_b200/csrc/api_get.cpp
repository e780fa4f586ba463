// C ABI of libdgrtm, part 5: getters (parity checks).  Everything leaves in the USER's element order.
#include <algorithm>

#include "ctx.h"

using namespace dgrtm;

namespace {
template <typename T, typename U> void copy_out(const std::vector<T>& v, U* out) {
  if (out) for (size_t i = 0; i < v.size(); ++i) out[i] = (U)v[i];
}
}  // namespace

extern "C" {

int dg_get_sizes(const dg_ctx* ctx, int64_t* K, int* Np, int* Nfp, int64_t* nbnd, int64_t* nr) {
  if (!ctx) return DG_ERR_ARG;
  if (K) *K = ctx->mesh.K;
  if (Np) *Np = ctx->Np;
  if (Nfp) *Nfp = ctx->Nfp;
  if (nbnd) *nbnd = (int64_t)ctx->mesh.bnd_k.size();
  if (nr) *nr = ctx->nr;
  return DG_OK;
}

int dg_get_nodes(const dg_ctx* ctx, double* r, double* s, double* t) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->re.r, r); copy_out(ctx->re.s, s); copy_out(ctx->re.t, t);
  return DG_OK;
}

int dg_get_operators(const dg_ctx* ctx, double* Dr, double* Ds, double* Dt, double* LIFT, int32_t* Fmask) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->re.Dr, Dr); copy_out(ctx->re.Ds, Ds); copy_out(ctx->re.Dt, Dt);
  copy_out(ctx->re.LIFT, LIFT); copy_out(ctx->re.Fmask, Fmask);
  return DG_OK;
}

int dg_get_connectivity(const dg_ctx* ctx, int32_t* EToE, int32_t* EToF, int32_t* mapP) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->mesh.EToE, EToE); copy_out(ctx->mesh.EToF, EToF); copy_out(ctx->mesh.mapP, mapP);
  return DG_OK;
}

int dg_get_boundary_faces(const dg_ctx* ctx, int32_t* bk, int32_t* bf, int32_t* bc) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->mesh.bnd_k, bk); copy_out(ctx->mesh.bnd_f, bf);
  if (bc)
    for (size_t b = 0; b < ctx->mesh.bnd_k.size(); ++b) bc[b] = ctx->mesh.bc[4 * (size_t)ctx->mesh.bnd_k[b] + ctx->mesh.bnd_f[b]];
  return DG_OK;
}

int dg_get_geometry(const dg_ctx* ctx, double* J, double* ginv, double* normals, double* gsur, double* ell) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->mesh.J, J); copy_out(ctx->mesh.ginv, ginv); copy_out(ctx->mesh.normals, normals);
  copy_out(ctx->mesh.gsur, gsur); copy_out(ctx->mesh.ell, ell);
  return DG_OK;
}

int dg_get_levels(const dg_ctx* ctx, int32_t* level) {
  if (!ctx || !level) return DG_ERR_ARG;
  if (!ctx->has_model) return DG_ERR_STATE;
  copy_out(ctx->model.level, level);
  return DG_OK;
}

int dg_get_dt(const dg_ctx* ctx, double* dt_local, int* nlocal) {
  if (!ctx) return DG_ERR_ARG;
  if (!ctx->has_model) return DG_ERR_STATE;
  if (dt_local) *dt_local = ctx->dt_local;
  if (nlocal) *nlocal = ctx->nlocal;
  return DG_OK;
}

int dg_get_time(const dg_ctx* ctx, double* t) {
  if (!ctx || !t) return DG_ERR_ARG;
  *t = ctx->t0 + (double)ctx->fine * ctx->dt_local;
  return DG_OK;
}

int dg_get_source(const dg_ctx* ctx, int32_t* k, double* w) {
  if (!ctx) return DG_ERR_ARG;
  if (!ctx->has_src) return DG_ERR_STATE;
  if (k) *k = (int32_t)ctx->src_k;
  copy_out(ctx->src_w, w);
  return DG_OK;
}

int dg_get_receivers(const dg_ctx* ctx, int32_t* k, double* rows, double* w) {
  if (!ctx) return DG_ERR_ARG;
  copy_out(ctx->rcv_k, k); copy_out(ctx->rcv_row, rows); copy_out(ctx->rcv_w, w);
  return DG_OK;
}

int dg_get_fields(dg_ctx* ctx, double* q) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!q) throw ApiError(DG_ERR_ARG, "q is NULL");
  fields_from_device(ctx, q, ctx->F.q);
  DG_CATCH(ctx)
}

int dg_get_traces(dg_ctx* ctx, double* qf) {
  DG_TRY(ctx)
  require_bound(ctx);
  if (!qf) throw ApiError(DG_ERR_ARG, "qf is NULL");
  const int Nfp = ctx->Nfp, REC = ctx->REC;
  std::vector<double> tmp((size_t)ctx->model.nslots * 4 * REC);
  normalize_traces(ctx, ctx->F);
  download_real(ctx, tmp.data(), ctx->F.qf, tmp.size());
  // device record (slot,f): [p | n.v][Nfp] at the READER's positions mapP[k][f][i]  ->  owner order
  for (int64_t s = 0; s < ctx->model.nslots; ++s) {
    const int64_t k = ctx->model.elem_of[s];
    if (k < 0) continue;
    for (int f = 0; f < 4; ++f) {
      const double* rec = &tmp[((size_t)s * 4 + f) * REC];
      const int32_t* mp = &ctx->mesh.mapP[((size_t)4 * k + f) * Nfp];
      for (int i = 0; i < Nfp; ++i) {
        qf[(((size_t)k * 4 + f) * Nfp + i) * 2 + 0] = rec[mp[i]];
        qf[(((size_t)k * 4 + f) * Nfp + i) * 2 + 1] = rec[Nfp + mp[i]];
      }
    }
  }
  DG_CATCH(ctx)
}

}  // extern "C"
