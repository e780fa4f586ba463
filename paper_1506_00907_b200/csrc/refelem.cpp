// Reference tetrahedron: warp-and-blend nodes, D_r/D_s/D_t, M^-1, L_f.
// PAPER.md:84-96 (nodal basis, N_p), PAPER.md:120 + App. A 593-612 (operators).  Node construction:
// DESIGN.md reading Q10.  Route: shifted monomials x^a y^b z^c on the unit simplex, closed-form Gram
// integrals a!b!c!/(a+b+c+3)!, all linear algebra in binary128 and rounded once to double.
#include "refelem.h"

#include <cmath>
#include <stdexcept>

namespace dgrtm {

typedef __float128 quad;

const int kFaceVertices[4][3] = {{0, 1, 2}, {0, 1, 3}, {1, 2, 3}, {0, 2, 3}};

namespace {

const double kAlphaOpt[7] = {0.0, 0.0, 0.0, 0.0, 0.1002, 1.1332, 1.5608};  // Warburton 2006 (Q10)

quad qabs(quad x) { return x < 0 ? -x : x; }

// inverse of an n x n matrix (row-major) by Gauss-Jordan with partial pivoting
std::vector<quad> inverse(std::vector<quad> A, int n) {
  std::vector<quad> B((size_t)n * n, 0);
  for (int i = 0; i < n; ++i) B[(size_t)i * n + i] = 1;
  for (int c = 0; c < n; ++c) {
    int p = c;
    for (int i = c + 1; i < n; ++i)
      if (qabs(A[(size_t)i * n + c]) > qabs(A[(size_t)p * n + c])) p = i;
    if (A[(size_t)p * n + c] == 0) throw std::runtime_error("singular matrix in reference element");
    if (p != c)
      for (int j = 0; j < n; ++j) {
        std::swap(A[(size_t)p * n + j], A[(size_t)c * n + j]);
        std::swap(B[(size_t)p * n + j], B[(size_t)c * n + j]);
      }
    quad piv = 1 / A[(size_t)c * n + c];
    for (int j = 0; j < n; ++j) {
      A[(size_t)c * n + j] *= piv;
      B[(size_t)c * n + j] *= piv;
    }
    for (int i = 0; i < n; ++i) {
      if (i == c) continue;
      quad f = A[(size_t)i * n + c];
      if (f == 0) continue;
      for (int j = 0; j < n; ++j) {
        A[(size_t)i * n + j] -= f * A[(size_t)c * n + j];
        B[(size_t)i * n + j] -= f * B[(size_t)c * n + j];
      }
    }
  }
  return B;
}

// C[n x m] = A[n x k] B[k x m]
std::vector<quad> matmul(const std::vector<quad>& A, const std::vector<quad>& B, int n, int k, int m) {
  std::vector<quad> C((size_t)n * m, 0);
  for (int i = 0; i < n; ++i)
    for (int l = 0; l < k; ++l) {
      quad a = A[(size_t)i * k + l];
      for (int j = 0; j < m; ++j) C[(size_t)i * m + j] += a * B[(size_t)l * m + j];
    }
  return C;
}

std::vector<quad> transpose(const std::vector<quad>& A, int n, int m) {
  std::vector<quad> T((size_t)n * m);
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < m; ++j) T[(size_t)j * n + i] = A[(size_t)i * m + j];
  return T;
}

quad ipow(quad x, int e) {
  quad p = 1;
  for (int i = 0; i < e; ++i) p *= x;
  return p;
}

quad factorial(int n) {
  quad f = 1;
  for (int i = 2; i <= n; ++i) f *= i;
  return f;
}

// Legendre P_n and P_n' at x
void legendre(int n, quad x, quad& P, quad& dP) {
  quad p0 = 1, p1 = x, d0 = 0, d1 = 1;
  if (n == 0) { P = 1; dP = 0; return; }
  for (int m = 1; m < n; ++m) {
    quad p2 = ((2 * m + 1) * x * p1 - m * p0) / (m + 1);
    quad d2 = ((2 * m + 1) * (p1 + x * d1) - m * d0) / (m + 1);
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  P = p1; dP = d1;
}

// Gauss-Lobatto-Legendre points on [-1,1], ascending: end points and the roots of P_N'
std::vector<quad> gauss_lobatto(int N) {
  std::vector<quad> g(N + 1);
  g[0] = -1; g[N] = 1;
  const double pi = 3.14159265358979323846;
  for (int i = 1; i < N; ++i) {
    quad x = -std::cos(pi * i / N);
    for (int it = 0; it < 60; ++it) {
      quad P, dP;
      legendre(N, x, P, dP);
      quad ddP = (2 * x * dP - (quad)N * (N + 1) * P) / (1 - x * x);   // Legendre ODE
      quad dx = dP / ddP;
      x -= dx;
      if (qabs(dx) < (quad)1e-30) break;
    }
    g[i] = x;
  }
  return g;
}

// displacement equispaced -> GLL, interpolated through the equispaced points, divided by 1-x^2
quad edge_warp(int N, const std::vector<quad>& gll, quad x) {
  quad w = 0;
  for (int i = 1; i < N; ++i) {
    quad ei = -1 + (quad)2 * i / N;
    quad term = (gll[i] - ei) / (1 - ei * ei);
    for (int j = 1; j < N; ++j) {
      if (j == i) continue;
      quad ej = -1 + (quad)2 * j / N;
      term *= (x - ej) / (ei - ej);
    }
    w += term;
  }
  return w;
}

}  // namespace

void build_reference_element(int N, RefElem& re) {
  if (N < 1 || N > 6) throw std::runtime_error("order N must be in 1..6");
  const int Np = (N + 1) * (N + 2) * (N + 3) / 6, Nfp = (N + 1) * (N + 2) / 2;
  re.N = N; re.Np = Np; re.Nfp = Nfp;

  // ---- nodes: equispaced barycentric lattice (r fastest, then s, then t), warped and blended
  re.lattice.assign((size_t)Np * 4, 0);
  std::vector<quad> lam((size_t)Np * 4);
  {
    int n = 0;
    for (int k = 0; k <= N; ++k)
      for (int j = 0; j <= N - k; ++j)
        for (int i = 0; i <= N - k - j; ++i, ++n) {
          int l[4] = {N - i - j - k, i, j, k};
          for (int v = 0; v < 4; ++v) {
            re.lattice[(size_t)n * 4 + v] = l[v];
            lam[(size_t)n * 4 + v] = (quad)l[v] / N;
          }
        }
  }
  const quad alpha = kAlphaOpt[N];
  const std::vector<quad> gll = gauss_lobatto(N);
  std::vector<quad> shift((size_t)Np * 4, 0);
  for (int a = 0; a < 4; ++a) {
    int o[3], c = 0;
    for (int v = 0; v < 4; ++v)
      if (v != a) o[c++] = v;
    const int edges[3][3] = {{o[0], o[1], o[2]}, {o[1], o[2], o[0]}, {o[2], o[0], o[1]}};
    for (int n = 0; n < Np; ++n) {
      const quad* L = &lam[(size_t)n * 4];
      const int* li = &re.lattice[(size_t)n * 4];
      quad fs[4] = {0, 0, 0, 0};
      for (int e = 0; e < 3; ++e) {
        int A = edges[e][0], B = edges[e][1], C = edges[e][2];
        quad amount = 2 * L[A] * L[B] * edge_warp(N, gll, L[B] - L[A]) * (1 + (alpha * L[C]) * (alpha * L[C]));
        fs[B] += amount;
        fs[A] -= amount;
      }
      quad la = L[a], lb = L[o[0]], lc = L[o[1]], ld = L[o[2]];
      quad blend = lb * lc * ld;
      quad denom = (lb + la / 2) * (lc + la / 2) * (ld + la / 2);
      if (denom > (quad)1e-10) blend = (1 + (alpha * la) * (alpha * la)) * blend / denom;
      for (int v = 0; v < 4; ++v) shift[(size_t)n * 4 + v] += blend * fs[v];
      // rim of face a (edges, vertices): the in-face warp alone (lattice integers: exact test)
      int npos = (li[o[0]] > 0) + (li[o[1]] > 0) + (li[o[2]] > 0);
      if (li[a] == 0 && npos < 3)
        for (int v = 0; v < 4; ++v) shift[(size_t)n * 4 + v] = fs[v];
    }
  }
  std::vector<quad> r(Np), s(Np), t(Np);
  re.r.resize(Np); re.s.resize(Np); re.t.resize(Np);
  for (int n = 0; n < Np; ++n) {
    quad l1 = lam[(size_t)n * 4 + 1] + shift[(size_t)n * 4 + 1];
    quad l2 = lam[(size_t)n * 4 + 2] + shift[(size_t)n * 4 + 2];
    quad l3 = lam[(size_t)n * 4 + 3] + shift[(size_t)n * 4 + 3];
    r[n] = -1 + 2 * l1; s[n] = -1 + 2 * l2; t[n] = -1 + 2 * l3;
    re.r[n] = (double)r[n]; re.s[n] = (double)s[n]; re.t[n] = (double)t[n];
  }

  // ---- shifted monomials x^a y^b z^c, x=(1+r)/2, ...: Vandermonde, derivatives, Gram matrix
  std::vector<int> ex;
  for (int a = 0; a <= N; ++a)
    for (int b = 0; b <= N - a; ++b)
      for (int c = 0; c <= N - a - b; ++c) { ex.push_back(a); ex.push_back(b); ex.push_back(c); }
  std::vector<quad> V((size_t)Np * Np), Vr(V.size()), Vs(V.size()), Vt(V.size()), G(V.size());
  for (int i = 0; i < Np; ++i) {
    quad x = (1 + r[i]) / 2, y = (1 + s[i]) / 2, z = (1 + t[i]) / 2;
    for (int m = 0; m < Np; ++m) {
      int a = ex[3 * m], b = ex[3 * m + 1], c = ex[3 * m + 2];
      V[(size_t)i * Np + m] = ipow(x, a) * ipow(y, b) * ipow(z, c);
      Vr[(size_t)i * Np + m] = a ? (quad)a / 2 * ipow(x, a - 1) * ipow(y, b) * ipow(z, c) : (quad)0;
      Vs[(size_t)i * Np + m] = b ? (quad)b / 2 * ipow(x, a) * ipow(y, b - 1) * ipow(z, c) : (quad)0;
      Vt[(size_t)i * Np + m] = c ? (quad)c / 2 * ipow(x, a) * ipow(y, b) * ipow(z, c - 1) : (quad)0;
    }
  }
  for (int m = 0; m < Np; ++m)
    for (int k = 0; k < Np; ++k) {
      int A = ex[3 * m] + ex[3 * k], B = ex[3 * m + 1] + ex[3 * k + 1], C = ex[3 * m + 2] + ex[3 * k + 2];
      // int over the bi-unit tet (volume 4/3 = 8 x unit simplex)
      G[(size_t)m * Np + k] = 8 * factorial(A) * factorial(B) * factorial(C) / factorial(A + B + C + 3);
    }
  std::vector<quad> Vinv = inverse(V, Np);
  std::vector<quad> Dr = matmul(Vr, Vinv, Np, Np, Np), Ds = matmul(Vs, Vinv, Np, Np, Np),
                    Dt = matmul(Vt, Vinv, Np, Np, Np);
  std::vector<quad> Ginv = inverse(G, Np);
  std::vector<quad> Minv = matmul(matmul(V, Ginv, Np, Np, Np), transpose(V, Np, Np), Np, Np, Np);

  auto to_double = [](const std::vector<quad>& A) {
    std::vector<double> d(A.size());
    for (size_t i = 0; i < A.size(); ++i) d[i] = (double)A[i];
    return d;
  };
  re.Dr = to_double(Dr); re.Ds = to_double(Ds); re.Dt = to_double(Dt);
  re.Minv = to_double(Minv);
  re.VinvT = to_double(transpose(Vinv, Np, Np));

  // ---- faces: Fmask from the lattice (exact), 2-D mass matrices, L_f = M^-1 E_f
  const int zero_coord[4] = {3, 2, 0, 1};      // barycentric coordinate that vanishes on face f
  re.Fmask.assign((size_t)4 * Nfp, 0);
  for (int f = 0; f < 4; ++f) {
    int c = 0;
    for (int n = 0; n < Np; ++n)
      if (re.lattice[(size_t)n * 4 + zero_coord[f]] == 0) re.Fmask[(size_t)f * Nfp + c++] = n;
    if (c != Nfp) throw std::runtime_error("face node count");
  }
  std::vector<int> ex2;
  for (int a = 0; a <= N; ++a)
    for (int b = 0; b <= N - a; ++b) { ex2.push_back(a); ex2.push_back(b); }
  std::vector<quad> G2((size_t)Nfp * Nfp);
  for (int m = 0; m < Nfp; ++m)
    for (int k = 0; k < Nfp; ++k) {
      int A = ex2[2 * m] + ex2[2 * k], B = ex2[2 * m + 1] + ex2[2 * k + 1];
      G2[(size_t)m * Nfp + k] = 4 * factorial(A) * factorial(B) / factorial(A + B + 2);  // area 2 = 4 x 1/2
    }
  std::vector<quad> LIFT((size_t)Np * 4 * Nfp, 0);
  for (int f = 0; f < 4; ++f) {
    std::vector<quad> V2((size_t)Nfp * Nfp);
    for (int i = 0; i < Nfp; ++i) {
      int n = re.Fmask[(size_t)f * Nfp + i];
      quad u = (f == 0 || f == 1) ? r[n] : s[n];
      quad v = (f == 0) ? s[n] : t[n];
      quad xi = (1 + u) / 2, eta = (1 + v) / 2;
      for (int m = 0; m < Nfp; ++m) V2[(size_t)i * Nfp + m] = ipow(xi, ex2[2 * m]) * ipow(eta, ex2[2 * m + 1]);
    }
    std::vector<quad> V2inv = inverse(V2, Nfp);
    std::vector<quad> M2 = matmul(matmul(transpose(V2inv, Nfp, Nfp), G2, Nfp, Nfp, Nfp), V2inv, Nfp, Nfp, Nfp);
    std::vector<quad> E((size_t)Np * Nfp, 0);
    for (int i = 0; i < Nfp; ++i)
      for (int j = 0; j < Nfp; ++j) E[(size_t)re.Fmask[(size_t)f * Nfp + i] * Nfp + j] = M2[(size_t)i * Nfp + j];
    std::vector<quad> Lf = matmul(Minv, E, Np, Np, Nfp);
    for (int n = 0; n < Np; ++n)
      for (int j = 0; j < Nfp; ++j) LIFT[(size_t)n * 4 * Nfp + f * Nfp + j] = Lf[(size_t)n * Nfp + j];
  }
  re.LIFT = to_double(LIFT);
}

void RefElem::interp_row(double r0, double s0, double t0, double* row) const {
  // l(r0) = V^-T phi(r0), phi = the shifted monomials
  std::vector<double> phi(Np);
  double x = 0.5 * (1 + r0), y = 0.5 * (1 + s0), z = 0.5 * (1 + t0);
  int m = 0;
  for (int a = 0; a <= N; ++a)
    for (int b = 0; b <= N - a; ++b)
      for (int c = 0; c <= N - a - b; ++c, ++m) phi[m] = std::pow(x, a) * std::pow(y, b) * std::pow(z, c);
  for (int n = 0; n < Np; ++n) {
    double acc = 0;
    for (int k = 0; k < Np; ++k) acc += VinvT[(size_t)n * Np + k] * phi[k];
    row[n] = acc;
  }
}

}  // namespace dgrtm
