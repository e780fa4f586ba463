// C ABI of libdgrtm, part 1: context, setup, device workspace (include/dgrtm.h).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <mutex>
#include <thread>

#include "ctx.h"

namespace dgrtm {

const KernelTable* dg_kernel_table_order1(int);
const KernelTable* dg_kernel_table_order2(int);
const KernelTable* dg_kernel_table_order3(int);
const KernelTable* dg_kernel_table_order4(int);
const KernelTable* dg_kernel_table_order5(int);
const KernelTable* dg_kernel_table_order6(int);

const KernelTable* get_kernel_table(int N, int precision) {
  switch (N) {
    case 1: return dg_kernel_table_order1(precision);
    case 2: return dg_kernel_table_order2(precision);
    case 3: return dg_kernel_table_order3(precision);
    case 4: return dg_kernel_table_order4(precision);
    case 5: return dg_kernel_table_order5(precision);
    case 6: return dg_kernel_table_order6(precision);
  }
  return nullptr;
}

// ---- Adams-Bashforth weights by exact polynomial integration (long double, rounded once) ---------
namespace {
typedef std::vector<long double> Poly;   // ascending coefficients
Poly pmul(const Poly& p, const Poly& q) {
  Poly o(p.size() + q.size() - 1, 0.0L);
  for (size_t i = 0; i < p.size(); ++i)
    for (size_t j = 0; j < q.size(); ++j) o[i + j] += p[i] * q[j];
  return o;
}
Poly pint(const Poly& p) {
  Poly o(p.size() + 1, 0.0L);
  for (size_t i = 0; i < p.size(); ++i) o[i + 1] = p[i] / (long double)(i + 1);
  return o;
}
long double peval(const Poly& p, long double x) {
  long double v = 0;
  for (size_t i = p.size(); i-- > 0;) v = v * x + p[i];
  return v;
}
// I_s = antiderivative of the Lagrange function l_s through the nodes 0, -1, .., -(order-1)
std::vector<Poly> ab_antiderivatives(int order) {
  std::vector<Poly> I;
  for (int s = 0; s < order; ++s) {
    Poly p(1, 1.0L);
    for (int j = 0; j < order; ++j) {
      if (j == s) continue;
      const long double xs = -(long double)s, xj = -(long double)j;
      p = pmul(p, Poly{-xj / (xs - xj), 1.0L / (xs - xj)});
    }
    I.push_back(pint(p));
  }
  return I;
}
}  // namespace

const AbCoef& ab_coef(int order) {
  static AbCoef tab[4];
  static std::once_flag once;
  std::call_once(once, [] {
    for (int m = 1; m <= 3; ++m) {
      AbCoef& c = tab[m];
      std::memset(&c, 0, sizeof(c));
      std::vector<Poly> I = ab_antiderivatives(m);
      for (int s = 0; s < m; ++s) {
        c.a[s] = (double)peval(I[s], 1.0L);                 // eq (18)
        c.b[s] = (double)peval(I[s], 0.5L);                 // eq (19)
        c.abar[s] = (double)peval(pint(I[s]), 1.0L);        // reading Q1(iii)
        for (int t = 0; t < m; ++t) c.C[3 * s + t] = (double)peval(pint(pmul(I[s], I[t])), 1.0L);  // (24)
      }
    }
    std::memset(&tab[0], 0, sizeof(AbCoef));
  });
  return tab[order < 0 ? 0 : (order > 3 ? 3 : order)];
}

void ab_partial(int order, double theta, double w[3]) {
  w[0] = w[1] = w[2] = 0;
  if (order < 1) return;
  std::vector<Poly> I = ab_antiderivatives(order > 3 ? 3 : order);
  for (size_t s = 0; s < I.size(); ++s) w[s] = (double)peval(I[s], (long double)theta);
}

double ricker(double t, double f0, double tp, double amp) {
  const double pi = 3.14159265358979323846;
  const double x = pi * f0 * (t - tp), a = x * x;
  return amp * (1.0 - 2.0 * a) * std::exp(-a);
}

// ---- small device helpers ------------------------------------------------------------------------
size_t field_bytes(const dg_ctx* c) { return (size_t)c->model.nslots * 4 * c->Np * c->rs; }
size_t trace_bytes(const dg_ctx* c) { return (size_t)c->model.nslots * 4 * c->REC * c->rs; }

void sync_stream(dg_ctx* c) { cuda_check(cudaStreamSynchronize(c->stream), "cudaStreamSynchronize"); }

void upload_raw(dg_ctx* c, void* dst, const void* src, size_t bytes) {
  if (!bytes) return;
  cuda_check(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream), "cudaMemcpyAsync H2D");
  sync_stream(c);
}

void upload_real(dg_ctx* c, void* dst, const double* src, size_t n) {
  if (!n) return;
  if (c->precision == 64) { upload_raw(c, dst, src, n * sizeof(double)); return; }
  std::vector<float> tmp(n);
  for (size_t i = 0; i < n; ++i) tmp[i] = (float)src[i];
  upload_raw(c, dst, tmp.data(), n * sizeof(float));
}

void download_real(dg_ctx* c, double* dst, const void* src, size_t n) {
  if (!n) return;
  if (c->precision == 64) {
    cuda_check(cudaMemcpyAsync(dst, src, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "cudaMemcpyAsync D2H");
    sync_stream(c);
    return;
  }
  std::vector<float> tmp(n);
  cuda_check(cudaMemcpyAsync(tmp.data(), src, n * sizeof(float), cudaMemcpyDeviceToHost, c->stream), "cudaMemcpyAsync D2H");
  sync_stream(c);
  for (size_t i = 0; i < n; ++i) dst[i] = (double)tmp[i];
}

// user order q[K][4][Np] <-> device [block][4Np][32], converted to / from the device precision in one pass,
// slots split over host threads (the e2e path: dg_set_state / dg_get_fields)
namespace {
template <typename F> void parallel_slots(int64_t ns, F body) {
  unsigned nt = std::thread::hardware_concurrency();
  nt = nt == 0 ? 1 : (nt > 16 ? 16 : nt);
  if (ns < 4096) nt = 1;
  std::vector<std::thread> th;
  const int64_t nb = (ns + 31) / 32, per = (nb + nt - 1) / nt;
  for (unsigned t = 0; t < nt; ++t) {
    const int64_t b0 = t * per, b1 = std::min<int64_t>(nb, b0 + per);
    if (b0 >= b1) break;
    th.emplace_back([=] { body(b0 * 32, std::min<int64_t>(ns, b1 * 32)); });
  }
  for (auto& x : th) x.join();
}
template <typename real> void pack_fields(const dg_ctx* c, real* out, const double* q) {
  const int W = 4 * c->Np;
  parallel_slots(c->model.nslots, [&](int64_t s0, int64_t s1) {
    for (int64_t s = s0; s < s1; ++s) {
      const int64_t k = c->model.elem_of[s], b = s >> 5, lane = s & 31;
      real* o = out + (size_t)b * W * 32 + lane;
      if (k < 0) { for (int x = 0; x < W; ++x) o[(size_t)x * 32] = 0; continue; }
      const double* in = q + (size_t)k * W;
      for (int x = 0; x < W; ++x) o[(size_t)x * 32] = (real)in[x];
    }
  });
}
template <typename real> void unpack_fields(const dg_ctx* c, double* q, const real* in) {
  const int W = 4 * c->Np;
  parallel_slots(c->model.nslots, [&](int64_t s0, int64_t s1) {
    for (int64_t s = s0; s < s1; ++s) {
      const int64_t k = c->model.elem_of[s], b = s >> 5, lane = s & 31;
      if (k < 0) continue;
      const real* i = in + (size_t)b * W * 32 + lane;
      double* o = q + (size_t)k * W;
      for (int x = 0; x < W; ++x) o[x] = (double)i[(size_t)x * 32];
    }
  });
}
}  // namespace

char* host_stage(dg_ctx* c, size_t bytes) {
  if (bytes > c->stage_bytes) {
    if (c->stage_host) cudaFreeHost(c->stage_host);
    c->stage_host = nullptr; c->stage_bytes = 0;
    cuda_check(cudaHostAlloc(reinterpret_cast<void**>(&c->stage_host), bytes, cudaHostAllocDefault), "cudaHostAlloc (staging)");
    c->stage_bytes = bytes;
  }
  return c->stage_host;
}

void fields_to_device(dg_ctx* c, char* dq, const double* q) {
  const size_t nbytes = (size_t)c->model.nslots * 4 * c->Np * c->rs;
  char* tmp = host_stage(c, nbytes);            // pinned: the copy runs at link speed, no hidden staging
  if (c->precision == 64) pack_fields(c, reinterpret_cast<double*>(tmp), q);
  else pack_fields(c, reinterpret_cast<float*>(tmp), q);
  upload_raw(c, dq, tmp, nbytes);
}

void fields_from_device(dg_ctx* c, double* q, const char* dq) {
  const size_t nbytes = (size_t)c->model.nslots * 4 * c->Np * c->rs;
  char* tmp = host_stage(c, nbytes);
  cuda_check(cudaMemcpyAsync(tmp, dq, nbytes, cudaMemcpyDeviceToHost, c->stream), "cudaMemcpyAsync D2H");
  sync_stream(c);
  if (c->precision == 64) unpack_fields(c, q, reinterpret_cast<const double*>(tmp));
  else unpack_fields(c, q, reinterpret_cast<const float*>(tmp));
}

// user order I[K][Np] <- device [block][Np][32], one threaded pass from the device precision
void image_from_device(dg_ctx* c, double* I, const char* dimg) {
  const int Np = c->Np;
  std::vector<char> tmp((size_t)c->model.nblocks * Np * 32 * c->rs);
  cuda_check(cudaMemcpyAsync(tmp.data(), dimg, tmp.size(), cudaMemcpyDeviceToHost, c->stream), "cudaMemcpyAsync D2H");
  sync_stream(c);
  const bool f64 = c->precision == 64;
  const char* base = tmp.data();
  parallel_slots(c->model.nslots, [&](int64_t s0, int64_t s1) {
    for (int64_t s = s0; s < s1; ++s) {
      const int64_t k = c->model.elem_of[s];
      if (k < 0) continue;
      const size_t o = (size_t)(s >> 5) * Np * 32 + (size_t)(s & 31);
      double* out = I + (size_t)k * Np;
      if (f64) { const double* in = reinterpret_cast<const double*>(base) + o; for (int n = 0; n < Np; ++n) out[n] = in[(size_t)n * 32]; }
      else { const float* in = reinterpret_cast<const float*>(base) + o; for (int n = 0; n < Np; ++n) out[n] = (double)in[(size_t)n * 32]; }
    }
  });
}

void clear_field(dg_ctx* c, Field& F) {
  cuda_check(cudaMemsetAsync(F.q, 0, field_bytes(c), c->stream), "memset q");
  for (int s = 0; s < 3; ++s) cuda_check(cudaMemsetAsync(F.hist[s], 0, field_bytes(c), c->stream), "memset hist");
  cuda_check(cudaMemsetAsync(F.qfb[0], 0, trace_bytes(c), c->stream), "memset qf");
  cuda_check(cudaMemsetAsync(F.qfb[1], 0, trace_bytes(c), c->stream), "memset qf");
  cuda_check(cudaMemsetAsync(F.qfh, 0, trace_bytes(c), c->stream), "memset qf");
  F.reset_history();
}

void refresh_traces(dg_ctx* c, Field& F) {
  // update kernel with zero weights: q unchanged, exposed traces rewritten (Alg. 4)
  UpdateArgs u;
  std::memset(&u, 0, sizeof(u));
  u.q = F.q; u.qf = F.qf; u.h0 = F.hist[0]; u.h1 = F.hist[1]; u.h2 = F.hist[2];
  u.geo = c->geo; u.wperm = c->wperm; u.blk0 = 0; u.nblk = (int)c->model.nblocks;
  u.c0 = u.c1 = u.c2 = 0; u.ops = c->ops;
  DG_LAUNCH(c, KC_UPDATE, c->kt->update(u, c->stream));
  for (int l = 0; l < kMaxLevels; ++l) F.par[l] = 0;
}

void normalize_traces(dg_ctx* c, Field& F) {
  const Model& md = c->model;
  const size_t per_slot = (size_t)4 * c->REC * c->rs;
  for (int l = 0; l < md.nlevels; ++l) {
    if (F.par[l] == 0 || md.lvl_nblk[l] == 0) { F.par[l] = 0; continue; }
    const size_t off = (size_t)md.lvl_blk0[l] * 32 * per_slot, n = (size_t)md.lvl_nblk[l] * 32 * per_slot;
    cuda_check(cudaMemcpyAsync(F.qfb[0] + off, F.qfb[1] + off, n, cudaMemcpyDeviceToDevice, c->stream), "normalize traces");
    F.par[l] = 0;
  }
}

}  // namespace dgrtm

using namespace dgrtm;

static thread_local std::string g_create_error;

extern "C" {

const char* dg_version(void) { return "dgrtm 0.1 (sm_100a)"; }

const char* dg_last_error(const dg_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int dg_mesh_create(dg_ctx** out, int N, int precision, int64_t K, int64_t Nv, const int32_t* EToV,
                   const double* VX, const int8_t* face_bc, int default_bc) {
  if (!out) { g_create_error = "out is NULL"; return DG_ERR_ARG; }
  *out = nullptr;
  if (!EToV || !VX || K <= 0 || Nv <= 0) { g_create_error = "NULL / empty mesh arrays"; return DG_ERR_ARG; }
  if (N < 1 || N > 6) { g_create_error = "order N must be in 1..6"; return DG_ERR_UNSUPPORTED; }
  if (precision != 32 && precision != 64) { g_create_error = "precision must be 32 or 64"; return DG_ERR_UNSUPPORTED; }
  if (default_bc < 1 || default_bc > 4) { g_create_error = "default_bc must be 1..4"; return DG_ERR_ARG; }
  if (K > (int64_t)500000000 / 4) { g_create_error = "too many elements for 32-bit face indices"; return DG_ERR_UNSUPPORTED; }
  dg_ctx* c = nullptr;
  try {
    c = new dg_ctx();
    c->N = N; c->precision = precision; c->rs = precision == 64 ? 8 : 4;
    build_reference_element(N, c->re);
    c->Np = c->re.Np; c->Nfp = c->re.Nfp; c->NF = 4 * c->Nfp; c->REC = 2 * c->Nfp;
    int64_t bad = -1;
    std::string msg = build_mesh(c->re, K, Nv, EToV, VX, face_bc, default_bc, c->mesh, &bad);
    if (!msg.empty()) {
      g_create_error = msg + " (element " + std::to_string(bad) + ")";
      delete c;
      return DG_ERR_MESH;
    }
    for (size_t i = 0; i < c->mesh.bc.size(); ++i)
      if (c->mesh.bc[i] == DG_BC_PRESCRIBED) c->has_prescribed = true;
    c->kt = get_kernel_table(N, precision);
    for (int l = 0; l < kMaxLevels; ++l) { c->d_stored[l] = nullptr; c->rec[l] = nullptr; }
    c->F.reset_history(); c->R.reset_history();
    if (const char* k = std::getenv("DGRTM_KERNEL")) { c->use_pipe = std::string(k) != "step"; c->use_tc = std::string(k) == "tc"; }
  } catch (const std::exception& e) {
    g_create_error = e.what();
    delete c;
    return DG_ERR_ARG;
  }
  *out = c;
  return DG_OK;
}

void dg_destroy(dg_ctx* ctx) { delete ctx; }
} // extern C
dg_ctx::~dg_ctx() {
  for (dgrtm::ProfEvent& e : prof_ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  for (int l = 0; l < dgrtm::kMaxLevels; ++l) {
    for (cudaEvent_t e : ev_step[l]) cudaEventDestroy(e);
    for (cudaEvent_t e : ev_copy[l]) cudaEventDestroy(e);
  }
  if (copy_stream) cudaStreamDestroy(copy_stream);
  if (stage_host) cudaFreeHost(stage_host);
}
extern "C" {

int dg_set_model(dg_ctx* ctx, const double* rho, const double* c, int nlevels, double cfl) {
  DG_TRY(ctx)
  if (!rho || !c) throw ApiError(DG_ERR_ARG, "rho / c is NULL");
  if (nlevels < 1 || nlevels > kMaxLevels) throw ApiError(DG_ERR_UNSUPPORTED, "nlevels must be in 1..8");
  if (!(cfl > 0)) throw ApiError(DG_ERR_ARG, "cfl must be positive");
  for (int64_t k = 0; k < ctx->mesh.K; ++k)
    if (!(rho[k] > 0) || !(c[k] > 0)) throw ApiError(DG_ERR_ARG, "rho and c must be positive (element " + std::to_string(k) + ")");
  build_model(ctx->re, ctx->mesh, rho, c, nlevels, cfl, ctx->model);
  ctx->dt_local = ctx->model.dt_local;
  ctx->nlocal = 1 << (nlevels - 1);
  ctx->has_model = true;
  ctx->bound = false; ctx->hist_bound = false;     // the slot layout changed
  DG_CATCH(ctx)
}

int dg_set_model_levels(dg_ctx* ctx, const double* rho, const double* c, int nlevels, double dt_local, const int32_t* level,
                        const int32_t* bnd_level) {
  DG_TRY(ctx)
  if (!rho || !c || !level) throw ApiError(DG_ERR_ARG, "rho / c / level is NULL");
  if (nlevels < 1 || nlevels > kMaxLevels) throw ApiError(DG_ERR_UNSUPPORTED, "nlevels must be in 1..8");
  if (!(dt_local > 0)) throw ApiError(DG_ERR_ARG, "dt_local must be positive");
  const Mesh& m = ctx->mesh;
  for (int64_t k = 0; k < m.K; ++k) {
    if (!(rho[k] > 0) || !(c[k] > 0)) throw ApiError(DG_ERR_ARG, "rho and c must be positive (element " + std::to_string(k) + ")");
    if (level[k] < 0 || level[k] >= nlevels) throw ApiError(DG_ERR_ARG, "level out of range (element " + std::to_string(k) + ")");
  }
  for (int64_t k = 0; k < m.K; ++k)
    for (int f = 0; f < 4; ++f) {     // eq (19) serves neighbours one level apart
      const int64_t k2 = m.EToE[4 * k + f];
      const int l2 = k2 >= 0 ? level[k2] : (bnd_level && m.bnd_index[4 * k + f] >= 0 ? bnd_level[m.bnd_index[4 * k + f]] : -1);
      if (l2 >= nlevels) throw ApiError(DG_ERR_ARG, "bnd_level out of range");
      if (l2 >= 0 && std::abs(l2 - level[k]) > 1) throw ApiError(DG_ERR_ARG, "face neighbours must be at most one level apart");
    }
  const ImposedLevels imp{dt_local, level, bnd_level};
  build_model(ctx->re, ctx->mesh, rho, c, nlevels, 1.0, ctx->model, &imp);
  ctx->dt_local = ctx->model.dt_local;
  ctx->nlocal = 1 << (nlevels - 1);
  ctx->has_model = true;
  ctx->bound = false; ctx->hist_bound = false;
  DG_CATCH(ctx)
}

int dg_set_integrator(dg_ctx* ctx, int integrator) {
  DG_TRY(ctx)
  if (integrator != DG_INTEGRATOR_AB3 && integrator != DG_INTEGRATOR_LSERK4) throw ApiError(DG_ERR_ARG, "unknown integrator");
  if (integrator == DG_INTEGRATOR_LSERK4 && ctx->has_model && ctx->model.nlevels != 1)
    throw ApiError(DG_ERR_UNSUPPORTED, "LSERK4 is single-rate only");
  if (integrator != ctx->integrator && ctx->bound) restart_history(ctx);
  ctx->integrator = integrator;
  DG_CATCH(ctx)
}

int dg_set_dt(dg_ctx* ctx, double dt_local) {
  DG_TRY(ctx)
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  if (!(dt_local > 0)) throw ApiError(DG_ERR_ARG, "dt_local must be positive");
  if (ctx->bound) restart_history(ctx);
  ctx->dt_local = dt_local;
  DG_CATCH(ctx)
}

} // extern C
namespace dgrtm {
// A change of integrator or step size invalidates the stored right-hand sides (LSERK4 uses hist[0] as stage scratch;
// AB weights assume equal spacing): the time base moves to the current time and AB restarts with AB1, AB2 (reading Q7).
void restart_history(dg_ctx* c) {
  normalize_traces(c, c->F);
  c->t0 = c->t0 + (double)c->fine * c->dt_local;
  c->fine = 0;
  c->F.reset_history();
}
}  // namespace dgrtm
extern "C" {

static void point_weights(dg_ctx* c, const double x[3], int64_t* k, double* row, double* w) {
  double rst[3];
  const int64_t e = c->locator.locate(c->mesh, x, rst);
  if (e < 0) throw ApiError(DG_ERR_ARG, "point outside the mesh");
  const int Np = c->Np;
  std::vector<double> ell(Np);
  c->re.interp_row(rst[0], rst[1], rst[2], ell.data());
  for (int n = 0; n < Np; ++n) {
    double acc = 0;
    for (int m = 0; m < Np; ++m) acc += c->re.Minv[(size_t)n * Np + m] * ell[m];
    w[n] = acc / c->mesh.J[e];                      // M_k^-1 l(x0), M_k = J_k M
    if (row) row[n] = ell[n];
  }
  *k = e;
}

int dg_set_source(dg_ctx* ctx, const double x0[3], int wavelet, double f0, double tp, double amp) {
  DG_TRY(ctx)
  if (!x0) throw ApiError(DG_ERR_ARG, "x0 is NULL");
  if (wavelet != DG_WAVELET_RICKER) throw ApiError(DG_ERR_UNSUPPORTED, "unknown wavelet");
  ctx->src_w.assign(ctx->Np, 0.0);
  point_weights(ctx, x0, &ctx->src_k, nullptr, ctx->src_w.data());
  ctx->f0 = f0; ctx->tp = tp; ctx->amp = amp;
  ctx->has_src = true;
  if (ctx->bound) { upload_real(ctx, ctx->d_src_w, ctx->src_w.data(), ctx->Np); upload_point_source(ctx); }
  DG_CATCH(ctx)
}

int dg_set_receivers(dg_ctx* ctx, int64_t nr, const double* xr) {
  DG_TRY(ctx)
  if (nr < 0 || (nr > 0 && !xr)) throw ApiError(DG_ERR_ARG, "bad receiver array");
  const int Np = ctx->Np;
  std::vector<int32_t> rk(nr);
  std::vector<double> row((size_t)nr * Np), w((size_t)nr * Np);
  for (int64_t r = 0; r < nr; ++r) {
    int64_t k;
    point_weights(ctx, xr + 3 * r, &k, &row[(size_t)r * Np], &w[(size_t)r * Np]);
    rk[r] = (int32_t)k;
  }
  ctx->nr = nr; ctx->rcv_k.swap(rk); ctx->rcv_row.swap(row); ctx->rcv_w.swap(w);
  // within the receiver capacity of the bound RTM region the region stays: image, q(t_f) and the trace history are
  // untouched and only the receiver tables are replaced (gathers of a survey stack in place)
  if (ctx->hist_bound && ctx->bound && nr <= ctx->nr_cap) upload_receiver_tables(ctx);
  else ctx->hist_bound = false;
  DG_CATCH(ctx)
}

// ---- workspace -------------------------------------------------------------------------------------
} // extern C
namespace dgrtm {
void carve_workspace(dg_ctx* c, Carver& cv) {
  const int Np = c->Np, Nfp = c->Nfp, NF = c->NF;
  const size_t rs = c->rs;
  const Model& md = c->model;
  c->ops.D3T = cv.take((size_t)3 * Np * Np * rs);
  c->ops.LIFTT = cv.take((size_t)NF * Np * rs);
  c->ops.Fmask = (const int*)cv.take((size_t)NF * 4);
  c->ops.nperm = (int)(c->mesh.ptab.size() / Nfp);
  c->ops.ptab = (const int*)cv.take(c->mesh.ptab.size() * 4);
  c->geo = cv.take((size_t)md.nblocks * DG_NGEO * 32 * rs);
  c->nbr = (int*)cv.take((size_t)md.nblocks * 4 * 32 * 4);
  c->wperm = (int*)cv.take((size_t)md.nblocks * 32 * 4);
  c->F.q = cv.take(field_bytes(c));
  for (int s = 0; s < 3; ++s) c->F.hist[s] = cv.take(field_bytes(c));
  c->F.qf = cv.take(trace_bytes(c));
  c->F.qfb[0] = c->F.qf;
  c->F.qfb[1] = cv.take(trace_bytes(c));
  c->F.qfh = cv.take(trace_bytes(c));
  {
    const int npad = c->kt ? c->kt->step_npad : Np;
    c->d_D3P = cv.take((size_t)3 * Np * npad * rs);
    c->d_LTP = cv.take((size_t)NF * npad * rs);
    c->d_D3Q = cv.take(std::max<size_t>(16, c->kt ? c->kt->pipe_blob_bytes : 0));
    c->d_LTQ = cv.take(std::max<size_t>(16, c->kt ? c->kt->tc_blob_bytes : 0));      // tensor-core kernel's tables
  }
  c->d_blkflag = (unsigned char*)cv.take((size_t)md.nblocks + 32);   // + the ticket counters (sched_counters)
  c->d_pt_src = (int*)cv.take((size_t)md.nslots * 4);
  c->scratch = cv.take(field_bytes(c));
  c->ext = cv.take(std::max<size_t>(1, c->mesh.bnd_k.size()) * Nfp * 2 * rs);
  c->d_src_w = cv.take((size_t)Np * rs);
  c->d_halo = cv.take(std::max<size_t>(1, c->mesh.bnd_k.size()) * (size_t)(4 + 8 + 4 * Nfp) + 64);   // halo tables (dg_set_halo)
  c->d_halo_face = cv.take(std::max<size_t>(1, c->mesh.bnd_k.size()) * (size_t)(8 + 4 + 4 * Nfp) + 64);   // the same by boundary face
  for (int l = 0; l < md.nlevels; ++l) {
    c->d_stored[l] = (int*)cv.take(std::max<size_t>(1, md.stored[l].size()) * 4);
  }
}
void check_launches(dg_ctx* c) {
  cuda_check(cudaGetLastError(), "kernel launch");
  if (c->kt && c->kt->take_error) {
    const int e = c->kt->take_error();
    if (e != 0) throw ApiError(DG_ERR_CUDA, std::string("cudaLaunchKernelEx: ") + cudaGetErrorString((cudaError_t)e));
  }
}
void require_bound(dg_ctx* c) {
  if (!c->bound) throw ApiError(DG_ERR_STATE, "no device workspace bound (dg_set_model, dg_workspace_bytes, dg_bind_workspace)");
}
}  // namespace dgrtm
extern "C" {

int dg_workspace_bytes(dg_ctx* ctx, size_t* n) {
  DG_TRY(ctx)
  if (!n) throw ApiError(DG_ERR_ARG, "n is NULL");
  if (!ctx->has_model) throw ApiError(DG_ERR_STATE, "dg_set_model first");
  Carver count;   // null base: only counts
  {
    // the carve writes pointers into the ctx: save and restore them so a bound ctx is not disturbed
    OpsDev ops = ctx->ops; char* geo = ctx->geo; int* nbr = ctx->nbr; int* wperm = ctx->wperm; Field F = ctx->F;
    char* scratch = ctx->scratch; char* ext = ctx->ext; char* sw = ctx->d_src_w; char* dh = ctx->d_halo;
    char* dp = ctx->d_D3P; char* lp = ctx->d_LTP; char* dq = ctx->d_D3Q; char* lq = ctx->d_LTQ; unsigned char* bf = ctx->d_blkflag; int* ps = ctx->d_pt_src;
    int* ds[kMaxLevels];
    for (int l = 0; l < kMaxLevels; ++l) ds[l] = ctx->d_stored[l];
    carve_workspace(ctx, count);
    ctx->ops = ops; ctx->geo = geo; ctx->nbr = nbr; ctx->wperm = wperm; ctx->F = F;
    ctx->scratch = scratch; ctx->ext = ext; ctx->d_src_w = sw; ctx->d_halo = dh;
    ctx->d_D3P = dp; ctx->d_LTP = lp; ctx->d_D3Q = dq; ctx->d_LTQ = lq; ctx->d_blkflag = bf; ctx->d_pt_src = ps;
    for (int l = 0; l < kMaxLevels; ++l) ctx->d_stored[l] = ds[l];
  }
  *n = count.used;
  DG_CATCH(ctx)
}

}  // extern "C"
