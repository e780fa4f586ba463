// Reference tetrahedron of the nodal DG scheme (host, built once per ctx).
// PAPER.md:84-96 (eqs (9)-(10), warp-and-blend nodes), PAPER.md:120 and App. A 593-612 (D_j, M, L_f).
#pragma once
#include <vector>

namespace dgrtm {

struct RefElem {
  int N = 0, Np = 0, Nfp = 0;
  std::vector<double> r, s, t;           // [Np]
  std::vector<int> lattice;              // [Np][4] integer barycentric lattice tuple of each node
  std::vector<double> Dr, Ds, Dt;        // [Np][Np]
  std::vector<double> Minv;              // [Np][Np] inverse reference mass matrix
  std::vector<double> LIFT;              // [Np][4*Nfp]
  std::vector<int> Fmask;                // [4][Nfp]
  // values of the Np Lagrange functions at a reference point
  void interp_row(double r0, double s0, double t0, double* row) const;
  std::vector<double> VinvT;             // [Np][Np]: (V^-1)^T for the shifted-monomial basis
};

// local faces as vertex triples: F0={0,1,2} (t=-1), F1={0,1,3} (s=-1), F2={1,2,3} (r+s+t=-1), F3={0,2,3} (r=-1)
extern const int kFaceVertices[4][3];

void build_reference_element(int N, RefElem& re);

}  // namespace dgrtm
