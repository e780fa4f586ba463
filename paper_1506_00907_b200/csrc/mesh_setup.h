// Host-side setup (fp64): geometry, connectivity, boundary faces, levels, device slot layout.
// PAPER.md:150-154 (levels), PAPER.md:258 (device tables), App. A PAPER.md:606-624 (geometry).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "refelem.h"

namespace dgrtm {

struct Mesh {
  int64_t K = 0, Nv = 0;
  std::vector<int32_t> EToV;        // [K][4]
  std::vector<double> VX;           // [Nv][3]
  std::vector<int32_t> EToE, EToF;  // [K][4], -1 on boundary
  std::vector<int32_t> mapP;        // [K][4][Nfp]
  std::vector<int8_t> bc;           // [K][4], 0 interior
  std::vector<int32_t> bnd_k, bnd_f;  // boundary-face list, ascending (k,f)
  std::vector<int32_t> bnd_index;   // [K][4] -> position in the list, -1 interior
  std::vector<double> J, ginv, normals, gsur, ell;  // [K], [K][9], [K][12], [K][4], [K]
  // unique face-node permutations (row 0 = identity) and the id of each (k,f)
  std::vector<int32_t> ptab;        // [nperm][Nfp]
  std::vector<uint8_t> perm_id;     // [K][4]
};

// returns "" or an error message; bad_elem receives the offending element (or -1)
std::string build_mesh(const RefElem& re, int64_t K, int64_t Nv, const int32_t* EToV, const double* VX,
                       const int8_t* face_bc, int default_bc, Mesh& m, int64_t* bad_elem);

struct Model {
  std::vector<double> rho, c, dt_k;
  double dt_local = 0;
  int nlevels = 1;
  std::vector<int32_t> level;             // [K] 0 = coarsest
  // slot layout: elements sorted by level (stable), every level padded to a multiple of 32
  int64_t nslots = 0, nblocks = 0;
  std::vector<int64_t> slot_of;           // [K]
  std::vector<int64_t> elem_of;           // [nslots], -1 = padding
  std::vector<int> lvl_blk0, lvl_nblk;    // per level
  std::vector<int64_t> lvl_count;         // real elements per level
  std::vector<std::vector<int32_t>> coarse_nb;   // per level: slots with a finer face neighbour
  std::vector<std::vector<int32_t>> stored;      // per level: boundary-list indices of absorbing faces
};

// levels and local step imposed from outside (a sub-domain takes those of the whole mesh, dg_set_model_levels);
// bnd_level[nbnd]: level of the element behind a boundary face in the neighbouring sub-domain, -1 = none (may be NULL)
struct ImposedLevels { double dt_local; const int32_t* level; const int32_t* bnd_level; };
void build_model(const RefElem& re, const Mesh& m, const double* rho, const double* c, int nlevels, double cfl,
                 Model& md, const ImposedLevels* imp = nullptr);

// element containing x (lowest id with all barycentrics >= -1e-10, reading Q11) and its (r,s,t); -1 if none.
// Candidates come from a uniform grid over the element bounding boxes, built on first use.
struct Locator {
  bool built = false;
  int n[3] = {1, 1, 1};
  double lo[3] = {0, 0, 0}, inv[3] = {0, 0, 0};
  std::vector<int64_t> start;
  std::vector<int32_t> items;
  int64_t locate(const Mesh& m, const double x[3], double rst[3]);
};

}  // namespace dgrtm
