// Host-side setup (fp64).  See mesh_setup.h.
#include "mesh_setup.h"

#include <algorithm>
#include <array>
#include <cmath>
#include <map>

namespace dgrtm {

namespace {

struct FaceKey {
  int32_t v[3];
  int32_t kf;
  bool operator<(const FaceKey& o) const {
    if (v[0] != o.v[0]) return v[0] < o.v[0];
    if (v[1] != o.v[1]) return v[1] < o.v[1];
    if (v[2] != o.v[2]) return v[2] < o.v[2];
    return kf < o.kf;
  }
  bool same(const FaceKey& o) const { return v[0] == o.v[0] && v[1] == o.v[1] && v[2] == o.v[2]; }
};

inline void cross(const double* a, const double* b, double* c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

}  // namespace

std::string build_mesh(const RefElem& re, int64_t K, int64_t Nv, const int32_t* EToV, const double* VX,
                       const int8_t* face_bc, int default_bc, Mesh& m, int64_t* bad_elem) {
  const int Nfp = re.Nfp, N = re.N;
  *bad_elem = -1;
  m.K = K; m.Nv = Nv;
  m.EToV.assign(EToV, EToV + 4 * K);
  m.VX.assign(VX, VX + 3 * Nv);
  for (int64_t i = 0; i < 4 * K; ++i)
    if (EToV[i] < 0 || EToV[i] >= Nv) { *bad_elem = i / 4; return "vertex index out of range"; }

  // ---- geometry of the affine map (App. A; g^vol = inverse Jacobian, reading Q3)
  m.J.resize(K); m.ginv.resize(9 * K); m.normals.resize(12 * K); m.gsur.resize(4 * K); m.ell.resize(K);
  for (int64_t k = 0; k < K; ++k) {
    const double* v0 = &VX[3 * EToV[4 * k]];
    const double* v1 = &VX[3 * EToV[4 * k + 1]];
    const double* v2 = &VX[3 * EToV[4 * k + 2]];
    const double* v3 = &VX[3 * EToV[4 * k + 3]];
    double xr[3], xs[3], xt[3], cst[3], ctr[3], crs[3];
    for (int d = 0; d < 3; ++d) { xr[d] = 0.5 * (v1[d] - v0[d]); xs[d] = 0.5 * (v2[d] - v0[d]); xt[d] = 0.5 * (v3[d] - v0[d]); }
    cross(xs, xt, cst); cross(xt, xr, ctr); cross(xr, xs, crs);
    const double J = xr[0] * cst[0] + xr[1] * cst[1] + xr[2] * cst[2];
    if (!(J > 0.0)) { *bad_elem = k; return "element with non-positive volume"; }
    m.J[k] = J;
    double gr[3], gs[3], gt[3];   // gradients of r, s, t
    for (int d = 0; d < 3; ++d) {
      gr[d] = cst[d] / J; gs[d] = ctr[d] / J; gt[d] = crs[d] / J;
      m.ginv[9 * k + 3 * d + 0] = gr[d]; m.ginv[9 * k + 3 * d + 1] = gs[d]; m.ginv[9 * k + 3 * d + 2] = gt[d];
    }
    double nv[4][3];
    for (int d = 0; d < 3; ++d) { nv[0][d] = -gt[d]; nv[1][d] = -gs[d]; nv[2][d] = gr[d] + gs[d] + gt[d]; nv[3][d] = -gr[d]; }
    const double volume = J * (4.0 / 3.0);
    double ell = 0;
    for (int f = 0; f < 4; ++f) {
      const double len = std::sqrt(nv[f][0] * nv[f][0] + nv[f][1] * nv[f][1] + nv[f][2] * nv[f][2]);
      m.gsur[4 * k + f] = len;                       // J_{k,f}/J_k
      for (int d = 0; d < 3; ++d) m.normals[12 * k + 3 * f + d] = nv[f][d] / len;
      const double area = 2.0 * len * J;
      const double h = 3.0 * volume / area;          // face-to-opposite-vertex distance
      if (f == 0 || h < ell) ell = h;
    }
    m.ell[k] = ell;
  }

  // ---- face connectivity: equal sorted vertex triples
  std::vector<FaceKey> keys((size_t)4 * K);
  for (int64_t k = 0; k < K; ++k)
    for (int f = 0; f < 4; ++f) {
      FaceKey& fk = keys[(size_t)4 * k + f];
      for (int j = 0; j < 3; ++j) fk.v[j] = EToV[4 * k + kFaceVertices[f][j]];
      std::sort(fk.v, fk.v + 3);
      if (fk.v[0] == fk.v[1] || fk.v[1] == fk.v[2]) { *bad_elem = k; return "element with repeated vertex"; }
      fk.kf = (int32_t)(4 * k + f);
    }
  std::sort(keys.begin(), keys.end());
  m.EToE.assign((size_t)4 * K, -1); m.EToF.assign((size_t)4 * K, -1);
  for (size_t i = 0; i + 1 < keys.size(); ++i) {
    if (!keys[i].same(keys[i + 1])) continue;
    if (i + 2 < keys.size() && keys[i].same(keys[i + 2])) {
      *bad_elem = keys[i].kf / 4;
      return "non-conforming mesh: a face is shared by more than two elements";
    }
    const int32_t a = keys[i].kf, b = keys[i + 1].kf;
    m.EToE[a] = b / 4; m.EToF[a] = b % 4;
    m.EToE[b] = a / 4; m.EToF[b] = a % 4;
    ++i;
  }

  // ---- face-node matching through the integer lattice (exact): weights of a face node on the
  // three face vertices identify it; the neighbour sees the same weights on the same global vertices
  std::vector<int> by_weights((size_t)4 * (N + 1) * (N + 1), -1);   // [f][w0][w1] -> face node
  for (int f = 0; f < 4; ++f)
    for (int i = 0; i < Nfp; ++i) {
      const int* l = &re.lattice[(size_t)re.Fmask[(size_t)f * Nfp + i] * 4];
      by_weights[((size_t)f * (N + 1) + l[kFaceVertices[f][0]]) * (N + 1) + l[kFaceVertices[f][1]]] = i;
    }
  m.mapP.resize((size_t)4 * K * Nfp);
  m.perm_id.assign((size_t)4 * K, 0);
  std::map<std::vector<int32_t>, int> perm_index;
  std::vector<int32_t> row(Nfp);
  for (int i = 0; i < Nfp; ++i) row[i] = i;
  perm_index[row] = 0;
  m.ptab = row;
  for (int64_t k = 0; k < K; ++k)
    for (int f = 0; f < 4; ++f) {
      int32_t* out = &m.mapP[((size_t)4 * k + f) * Nfp];
      const int64_t k2 = m.EToE[4 * k + f];
      if (k2 < 0) {
        for (int i = 0; i < Nfp; ++i) out[i] = i;
        continue;
      }
      const int f2 = m.EToF[4 * k + f];
      int sigma[3];   // neighbour face vertex j2 -> my face vertex j
      for (int j2 = 0; j2 < 3; ++j2) {
        const int32_t g = EToV[4 * k2 + kFaceVertices[f2][j2]];
        sigma[j2] = -1;
        for (int j = 0; j < 3; ++j)
          if (EToV[4 * k + kFaceVertices[f][j]] == g) sigma[j2] = j;
      }
      for (int i = 0; i < Nfp; ++i) {
        const int* l = &re.lattice[(size_t)re.Fmask[(size_t)f * Nfp + i] * 4];
        const int wmine[3] = {l[kFaceVertices[f][0]], l[kFaceVertices[f][1]], l[kFaceVertices[f][2]]};
        out[i] = by_weights[((size_t)f2 * (N + 1) + wmine[sigma[0]]) * (N + 1) + wmine[sigma[1]]];
      }
      for (int i = 0; i < Nfp; ++i) row[i] = out[i];
      auto it = perm_index.find(row);
      if (it == perm_index.end()) {
        const int id = (int)perm_index.size();
        if (id >= 32) return "more than 32 distinct face permutations";
        perm_index[row] = id;
        m.ptab.insert(m.ptab.end(), row.begin(), row.end());
        m.perm_id[4 * k + f] = (uint8_t)id;
      } else {
        m.perm_id[4 * k + f] = (uint8_t)it->second;
      }
    }

  // ---- boundary faces
  m.bc.assign((size_t)4 * K, 0);
  m.bnd_index.assign((size_t)4 * K, -1);
  m.bnd_k.clear(); m.bnd_f.clear();
  for (int64_t k = 0; k < K; ++k)
    for (int f = 0; f < 4; ++f) {
      if (m.EToE[4 * k + f] >= 0) continue;
      int t = face_bc ? face_bc[4 * k + f] : 0;
      if (t <= 0) t = default_bc;
      if (t < 1 || t > 4) { *bad_elem = k; return "boundary-condition type must be 1..4"; }
      m.bc[4 * k + f] = (int8_t)t;
      m.bnd_index[4 * k + f] = (int32_t)m.bnd_k.size();
      m.bnd_k.push_back((int32_t)k); m.bnd_f.push_back(f);
    }
  return "";
}

void build_model(const RefElem& re, const Mesh& m, const double* rho, const double* c, int nlevels, double cfl,
                 Model& md, const ImposedLevels* imp) {
  const int64_t K = m.K;
  const int N = re.N, L = nlevels;
  md.rho.assign(rho, rho + K); md.c.assign(c, c + K);
  md.nlevels = L;
  // local stable step (eq (17))
  md.dt_k.resize(K);
  double dtmin = 0;
  for (int64_t k = 0; k < K; ++k) {
    md.dt_k[k] = cfl * m.ell[k] / ((double)((N + 1) * (N + 1)) * c[k]);
    if (k == 0 || md.dt_k[k] < dtmin) dtmin = md.dt_k[k];
  }
  md.dt_local = dtmin;
  // raw exponent j = max{ j <= L-1 : 2^j dt_local <= dt_k }, then lowered so that face neighbours
  // differ by at most one (reading Q9); bucket propagation from the finest values up
  std::vector<int> j(K, 0);
  for (int64_t k = 0; k < K; ++k)
    for (int e = 1; e < L; ++e)
      if (std::ldexp(dtmin, e) <= md.dt_k[k]) j[k] = e;
  std::vector<std::vector<int64_t>> bucket(L);
  for (int64_t k = 0; k < K; ++k) bucket[j[k]].push_back(k);
  for (int val = 0; val + 1 < L; ++val)
    for (size_t x = 0; x < bucket[val].size(); ++x) {
      const int64_t k = bucket[val][x];
      if (j[k] != val) continue;
      for (int f = 0; f < 4; ++f) {
        const int64_t k2 = m.EToE[4 * k + f];
        if (k2 >= 0 && j[k2] > val + 1) { j[k2] = val + 1; bucket[val + 1].push_back(k2); }
      }
    }
  md.level.resize(K);
  for (int64_t k = 0; k < K; ++k) md.level[k] = (L - 1) - j[k];
  if (imp) {   // a sub-domain of a decomposition: the levels and the step of the WHOLE mesh (dg_set_model_levels)
    md.dt_local = imp->dt_local;
    for (int64_t k = 0; k < K; ++k) md.level[k] = imp->level[k];
  }
  // level of the element behind a boundary face in the neighbouring sub-domain (-1: none)
  auto outer_level = [&](int64_t k, int f) -> int {
    if (!imp || !imp->bnd_level) return -1;
    const int32_t b = m.bnd_index[4 * k + f];
    return b < 0 ? -1 : imp->bnd_level[b];
  };

  // ---- slot layout
  md.lvl_blk0.assign(L, 0); md.lvl_nblk.assign(L, 0); md.lvl_count.assign(L, 0);
  for (int64_t k = 0; k < K; ++k) md.lvl_count[md.level[k]]++;
  int blk = 0;
  std::vector<int64_t> next(L);
  for (int l = 0; l < L; ++l) {
    md.lvl_blk0[l] = blk;
    md.lvl_nblk[l] = (int)((md.lvl_count[l] + 31) / 32);
    next[l] = (int64_t)blk * 32;
    blk += md.lvl_nblk[l];
  }
  md.nblocks = blk; md.nslots = (int64_t)blk * 32;
  md.slot_of.resize(K); md.elem_of.assign(md.nslots, -1);
  // within a level: first the elements with a finer face neighbour (they expose half-step traces, eq (19)), then
  // the others, each in ascending element order - the blocks that need the second trace pass are as few as possible
  auto has_finer = [&](int64_t k) {
    for (int f = 0; f < 4; ++f) {
      const int64_t k2 = m.EToE[4 * k + f];
      if (k2 >= 0 && md.level[k2] > md.level[k]) return true;
      if (k2 < 0 && outer_level(k, f) > md.level[k]) return true;
    }
    return false;
  };
  for (int pass = 0; pass < 2; ++pass)
    for (int64_t k = 0; k < K; ++k) {
      if (has_finer(k) != (pass == 0)) continue;
      const int64_t s = next[md.level[k]]++;
      md.slot_of[k] = s; md.elem_of[s] = k;
    }
  // ---- elements with a finer neighbour (coarse neighbours of Alg. 1)
  md.coarse_nb.assign(L, {});
  for (int l = 0; l < L; ++l)
    for (int64_t s = (int64_t)md.lvl_blk0[l] * 32; s < (int64_t)(md.lvl_blk0[l] + md.lvl_nblk[l]) * 32; ++s) {
      const int64_t k = md.elem_of[s];
      if (k < 0) continue;
      bool finer = false;
      for (int f = 0; f < 4; ++f) {
        const int64_t k2 = m.EToE[4 * k + f];
        if (k2 >= 0 && md.level[k2] > md.level[k]) finer = true;
        if (k2 < 0 && outer_level(k, f) > md.level[k]) finer = true;
      }
      if (finer) md.coarse_nb[l].push_back((int32_t)s);
    }
  // ---- stored (absorbing) boundary faces per level, ascending boundary-list order (reading Q12)
  md.stored.assign(L, {});
  for (size_t b = 0; b < m.bnd_k.size(); ++b)
    if (m.bc[4 * (size_t)m.bnd_k[b] + m.bnd_f[b]] == 2) md.stored[md.level[m.bnd_k[b]]].push_back((int32_t)b);
}

int64_t Locator::locate(const Mesh& m, const double x[3], double rst[3]) {
  // uniform grid over the vertex bounding box, built on first use
  Locator& g = *this;
  const int64_t K = m.K;
  auto cell_range = [&](const double* bl, const double* bh, int* c0, int* c1) {
    for (int d = 0; d < 3; ++d) {
      c0[d] = std::max(0, std::min(g.n[d] - 1, (int)std::floor((bl[d] - g.lo[d]) * g.inv[d])));
      c1[d] = std::max(0, std::min(g.n[d] - 1, (int)std::floor((bh[d] - g.lo[d]) * g.inv[d])));
    }
  };
  if (!g.built) {
    g.built = true;
    double hi[3];
    for (int d = 0; d < 3; ++d) { g.lo[d] = 1e300; hi[d] = -1e300; }
    for (int64_t v = 0; v < m.Nv; ++v)
      for (int d = 0; d < 3; ++d) { g.lo[d] = std::min(g.lo[d], m.VX[3 * v + d]); hi[d] = std::max(hi[d], m.VX[3 * v + d]); }
    const double cells = std::max(1.0, (double)K / 6.0);
    const double vol = std::max(1e-300, (hi[0] - g.lo[0]) * (hi[1] - g.lo[1]) * (hi[2] - g.lo[2]));
    const double h = std::cbrt(vol / cells);
    for (int d = 0; d < 3; ++d) {
      g.n[d] = std::max(1, std::min(256, (int)std::ceil((hi[d] - g.lo[d]) / h)));
      g.inv[d] = g.n[d] / std::max(1e-300, hi[d] - g.lo[d]);
    }
    const size_t ncell = (size_t)g.n[0] * g.n[1] * g.n[2];
    std::vector<int64_t> count(ncell + 1, 0);
    for (int pass = 0; pass < 2; ++pass) {
      for (int64_t k = 0; k < K; ++k) {
        double bl[3] = {1e300, 1e300, 1e300}, bh[3] = {-1e300, -1e300, -1e300};
        for (int v = 0; v < 4; ++v)
          for (int d = 0; d < 3; ++d) {
            const double xv = m.VX[3 * (size_t)m.EToV[4 * k + v] + d];
            bl[d] = std::min(bl[d], xv); bh[d] = std::max(bh[d], xv);
          }
        int c0[3], c1[3];
        cell_range(bl, bh, c0, c1);
        for (int a = c0[0]; a <= c1[0]; ++a)
          for (int b = c0[1]; b <= c1[1]; ++b)
            for (int c = c0[2]; c <= c1[2]; ++c) {
              const size_t cell = ((size_t)a * g.n[1] + b) * g.n[2] + c;
              if (pass == 0) count[cell + 1]++;
              else g.items[count[cell]++] = (int32_t)k;
            }
      }
      if (pass == 0) {
        for (size_t i = 0; i < ncell; ++i) count[i + 1] += count[i];
        g.start = count;
        g.items.resize((size_t)count[ncell]);
        count.assign(g.start.begin(), g.start.end());
      }
    }
  }
  int c0[3], c1[3];
  cell_range(x, x, c0, c1);
  const size_t cell = ((size_t)c0[0] * g.n[1] + c0[1]) * g.n[2] + c0[2];
  int64_t best = -1;
  for (int64_t it = g.start[cell]; it < g.start[cell + 1]; ++it) {
    const int64_t k = g.items[it];
    if (best >= 0 && k > best) continue;
    const double* v0 = &m.VX[3 * (size_t)m.EToV[4 * k]];
    const double d[3] = {x[0] - v0[0], x[1] - v0[1], x[2] - v0[2]};
    double q[3];   // (1+r, 1+s, 1+t)
    for (int jj = 0; jj < 3; ++jj)
      q[jj] = m.ginv[9 * k + jj] * d[0] + m.ginv[9 * k + 3 + jj] * d[1] + m.ginv[9 * k + 6 + jj] * d[2];
    const double l0 = 1.0 - 0.5 * (q[0] + q[1] + q[2]);
    if (l0 >= -1e-10 && 0.5 * q[0] >= -1e-10 && 0.5 * q[1] >= -1e-10 && 0.5 * q[2] >= -1e-10) {
      best = k;
      rst[0] = q[0] - 1.0; rst[1] = q[1] - 1.0; rst[2] = q[2] - 1.0;
    }
  }
  return best;
}

}  // namespace dgrtm
