"""ORACLE (test infrastructure, fp64, plain numpy) - reference tetrahedron of the nodal DG scheme.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package; the CUDA path shares no code with it.

What is computed (PAPER.md = /root/reference/PAPER.md):
  * nodes: N_p = (N+1)(N+2)(N+3)/6 warp-and-blend nodes (eq. (9)-(10) context;
    construction per Warburton 2006 as read in DESIGN.md reading Q10 - the exact nodes of the paper
    are "parity unpinned", only their properties are pinned in tests/test_oracle_operators.py)
  * D_j (differentiation matrices), M (mass), L_f (lifting matrices)  (App. A 593-612)

Construction route (deliberately different from the CUDA library's host setup, which uses monomials
with closed-form Gram integrals in extended precision): an orthogonal collapsed-Jacobi basis written
homogeneously (no singular coordinates), integrals by a collapsed-coordinate Gauss-Jacobi rule.

Reference element: r,s,t >= -1, r+s+t <= -1; vertices v0=(-1,-1,-1), v1=(1,-1,-1), v2=(-1,1,-1),
v3=(-1,-1,1).  Local faces (vertex sets): F0={0,1,2} (t=-1), F1={0,1,3} (s=-1), F2={1,2,3}
(r+s+t=-1), F3={0,2,3} (r=-1).  Node order: equispaced-lattice order, r fastest, then s, then t.
"""
from dataclasses import dataclass

import numpy as np
from numpy.polynomial import legendre as npleg
from scipy.special import roots_jacobi

FACE_VERTICES = ((0, 1, 2), (0, 1, 3), (1, 2, 3), (0, 2, 3))
# optimised blend parameter alpha_N of Warburton (2006), N = 1..6 (reading Q10)
ALPHA_OPT = {1: 0.0, 2: 0.0, 3: 0.0, 4: 0.1002, 5: 1.1332, 6: 1.5608}


def num_nodes(N):
    return (N + 1) * (N + 2) * (N + 3) // 6


def num_face_nodes(N):
    return (N + 1) * (N + 2) // 2


# ------------------------------------------------------------------------------------------------
# 1-D ingredients
# ------------------------------------------------------------------------------------------------
def gauss_lobatto_nodes(N):
    """Gauss-Lobatto-Legendre points on [-1,1], ascending: the end points and the roots of P_N'."""
    if N == 1:
        return np.array([-1.0, 1.0])
    coef = np.zeros(N + 1)
    coef[N] = 1.0
    interior = npleg.legroots(npleg.legder(coef))
    return np.concatenate([[-1.0], np.sort(interior.real), [1.0]])


def edge_warp(N, x):
    """w(x) = [sum_i (g_i - e_i) l_i^e(x)] / (1 - x^2): displacement that carries the equispaced
    points e_i onto the Gauss-Lobatto points g_i, interpolated through the equispaced points and
    divided by the edge bubble 1-x^2 (the end-point factors are cancelled analytically)."""
    x = np.asarray(x, dtype=np.float64)
    e = np.linspace(-1.0, 1.0, N + 1)
    g = gauss_lobatto_nodes(N)
    w = np.zeros_like(x)
    for i in range(1, N):
        term = np.full_like(x, (g[i] - e[i]) / (1.0 - e[i] * e[i]))
        for j in range(1, N):
            if j != i:
                term = term * (x - e[j]) / (e[i] - e[j])
        w += term
    return w


# ------------------------------------------------------------------------------------------------
# nodes
# ------------------------------------------------------------------------------------------------
def equispaced_barycentric(N):
    """Barycentric coordinates [Np,4] (w.r.t. v0..v3) of the equispaced lattice, r fastest."""
    lam = []
    for k in range(N + 1):
        for j in range(N + 1 - k):
            for i in range(N + 1 - k - j):
                lam.append([(N - i - j - k) / N, i / N, j / N, k / N])
    return np.array(lam, dtype=np.float64)


def warp_blend_nodes(N, alpha=None):
    """Warp-and-blend nodes, formulated directly in barycentric coordinates.

    For the face opposite vertex a (vertices b,c,d) the in-face warp moves barycentric mass along
    each of its three edges (A,B), third face vertex C:
        d_AB = 2 lam_A lam_B w(lam_B - lam_A) (1 + (alpha lam_C)^2),  lam_B += d_AB, lam_A -= d_AB
    and is blended into the volume with
        lam_b lam_c lam_d (1 + (alpha lam_a)^2) / ((lam_b+lam_a/2)(lam_c+lam_a/2)(lam_d+lam_a/2)).
    Nodes on the rim of a face take that face's in-face warp alone (there the blend is 0/0)."""
    if alpha is None:
        alpha = ALPHA_OPT[N]
    lam = equispaced_barycentric(N)
    tol = 1e-10
    shift = np.zeros_like(lam)
    for a in range(4):
        b, c, d = [v for v in range(4) if v != a]
        face_shift = np.zeros_like(lam)
        for (A, B, C) in ((b, c, d), (c, d, b), (d, b, c)):
            amount = (2.0 * lam[:, A] * lam[:, B] * edge_warp(N, lam[:, B] - lam[:, A])
                      * (1.0 + (alpha * lam[:, C]) ** 2))
            face_shift[:, B] += amount
            face_shift[:, A] -= amount
        la, lb, lc, ld = lam[:, a], lam[:, b], lam[:, c], lam[:, d]
        blend = lb * lc * ld
        denom = (lb + 0.5 * la) * (lc + 0.5 * la) * (ld + 0.5 * la)
        ok = denom > tol
        blend[ok] = (1.0 + (alpha * la[ok]) ** 2) * blend[ok] / denom[ok]
        shift += blend[:, None] * face_shift
        rim = (la < tol) & (((lb > tol).astype(int) + (lc > tol) + (ld > tol)) < 3)
        shift[rim] = face_shift[rim]
    lam = lam + shift
    rst = -1.0 + 2.0 * lam[:, 1:4]
    return rst[:, 0].copy(), rst[:, 1].copy(), rst[:, 2].copy()


# ------------------------------------------------------------------------------------------------
# basis, quadrature
# ------------------------------------------------------------------------------------------------
def _multi_indices(N, dim):
    if dim == 3:
        return [(a, b, c) for a in range(N + 1) for b in range(N + 1 - a) for c in range(N + 1 - a - b)]
    return [(a, b) for a in range(N + 1) for b in range(N + 1 - a)]


def homogeneous_jacobi(n, alpha, X, S):
    """H_n(X,S) = S^n P_n^{(alpha,0)}(2X/S - 1) and its partial derivatives (dH/dX, dH/dS).

    P_n^{(alpha,0)} is the (unnormalised) Jacobi polynomial; written homogeneously in (X,S) the
    collapsed-coordinate singularity of the simplex basis disappears (H_n is a polynomial in X and
    S).  Three-term recurrence with S*x = 2X - S, differentiated term by term (forward mode):
      2(m+1)(m+a+1)(2m+a) P_{m+1} = (2m+a+1)[(2m+a+2)(2m+a) x + a^2] P_m - 2m(m+a)(2m+a+2) P_{m-1}.
    """
    X = np.asarray(X, dtype=np.float64)
    S = np.asarray(S, dtype=np.float64) + 0.0 * X
    X = X + 0.0 * S
    one, zero = np.ones_like(X), np.zeros_like(X)
    if n == 0:
        return one, zero, zero
    a = float(alpha)
    # P_1 = ((a+2) x + a)/2  ->  H_1 = ((a+2)(2X - S) + a S)/2
    Hm, Hm_X, Hm_S = one, zero, zero
    H = 0.5 * ((a + 2.0) * (2.0 * X - S) + a * S)
    H_X = (a + 2.0) * one
    H_S = -one
    for m in range(1, n):
        c1 = 2.0 * (m + 1) * (m + a + 1) * (2 * m + a)
        c2 = (2 * m + a + 1) * (2 * m + a + 2) * (2 * m + a)
        c3 = (2 * m + a + 1) * a * a
        c4 = 2.0 * m * (m + a) * (2 * m + a + 2)
        L = c2 * (2.0 * X - S) + c3 * S
        Hn = (L * H - c4 * S * S * Hm) / c1
        Hn_X = (2.0 * c2 * H + L * H_X - c4 * S * S * Hm_X) / c1
        Hn_S = ((c3 - c2) * H + L * H_S - c4 * (2.0 * S * Hm + S * S * Hm_S)) / c1
        Hm, Hm_X, Hm_S = H, H_X, H_S
        H, H_X, H_S = Hn, Hn_X, Hn_S
    return H, H_X, H_S


def simplex_basis(N, r, s, t, grad=False):
    """Orthogonal polynomial basis of P_N on the reference tet, evaluated at points (r,s,t):
        psi_ijk = F_i(x, sigma) G_ij(y, tau) H_ijk(t),   i+j+k <= N,
        F_i  = sigma^i P_i^{(0,0)}(2x/sigma - 1),        x = (1+r)/2, sigma = -(s+t)/2,
        G_ij = tau^j  P_j^{(2i+1,0)}(2y/tau - 1),        y = (1+s)/2, tau = (1-t)/2,
        H_ijk = P_k^{(2i+2j+2,0)}(t).
    (Collapsed-coordinate Jacobi products written as polynomials; unnormalised.)  With grad also the
    r, s, t derivatives by the chain rule (dx/dr = dy/ds = 1/2, dsigma/ds = dsigma/dt = dtau/dt = -1/2)."""
    r, s, t = (np.asarray(v, dtype=np.float64) for v in (r, s, t))
    x, sigma, y, tau = 0.5 * (1 + r), -0.5 * (s + t), 0.5 * (1 + s), 0.5 * (1 - t)
    idx = _multi_indices(N, 3)
    V = np.empty((len(r), len(idx)))
    if grad:
        Vr, Vs, Vt = np.empty_like(V), np.empty_like(V), np.empty_like(V)
    for m, (i, j, k) in enumerate(idx):
        F, F_x, F_sig = homogeneous_jacobi(i, 0, x, sigma)
        G, G_y, G_tau = homogeneous_jacobi(j, 2 * i + 1, y, tau)
        H, H_X, _ = homogeneous_jacobi(k, 2 * i + 2 * j + 2, 0.5 * (1 + t), 1.0)
        V[:, m] = F * G * H
        if grad:
            Vr[:, m] = 0.5 * F_x * G * H
            Vs[:, m] = -0.5 * F_sig * G * H + 0.5 * F * G_y * H
            Vt[:, m] = -0.5 * F_sig * G * H - 0.5 * F * G_tau * H + F * G * (0.5 * H_X)
    return (V, Vr, Vs, Vt) if grad else V


def triangle_basis(N, u, v):
    """Orthogonal basis of P_N on the reference triangle: F_i((1+u)/2, (1-v)/2) P_j^{(2i+1,0)}(v)."""
    u, v = np.asarray(u, dtype=np.float64), np.asarray(v, dtype=np.float64)
    idx = _multi_indices(N, 2)
    V = np.empty((len(u), len(idx)))
    for m, (i, j) in enumerate(idx):
        F, _, _ = homogeneous_jacobi(i, 0, 0.5 * (1 + u), 0.5 * (1 - v))
        G, _, _ = homogeneous_jacobi(j, 2 * i + 1, 0.5 * (1 + v), 1.0)
        V[:, m] = F * G
    return V


def tet_quadrature(n):
    """Collapsed-coordinate Gauss rule on the reference tet, exact for total degree <= 2n-1.
    r = (1+a)(1-b)(1-c)/4 - 1, s = (1+b)(1-c)/2 - 1, t = c; dV = (1-b)/2 ((1-c)/2)^2 da db dc."""
    xa, wa = roots_jacobi(n, 0.0, 0.0)
    xb, wb = roots_jacobi(n, 1.0, 0.0)     # weight (1-b)
    xc, wc = roots_jacobi(n, 2.0, 0.0)     # weight (1-c)^2
    A, B, C = np.meshgrid(xa, xb, xc, indexing="ij")
    W = wa[:, None, None] * wb[None, :, None] * wc[None, None, :] / 8.0
    r = (1 + A) * (1 - B) * (1 - C) / 4 - 1
    s = (1 + B) * (1 - C) / 2 - 1
    return r.ravel(), s.ravel(), C.ravel(), W.ravel()


def tri_quadrature(n):
    """Collapsed Gauss rule on the reference triangle u,v >= -1, u+v <= 0 (area 2)."""
    xa, wa = roots_jacobi(n, 0.0, 0.0)
    xb, wb = roots_jacobi(n, 1.0, 0.0)
    A, B = np.meshgrid(xa, xb, indexing="ij")
    W = wa[:, None] * wb[None, :] / 2.0
    u = (1 + A) * (1 - B) / 2 - 1
    return u.ravel(), B.ravel(), W.ravel()


# ------------------------------------------------------------------------------------------------
# the reference element
# ------------------------------------------------------------------------------------------------
@dataclass
class ReferenceElement:
    N: int
    Np: int
    Nfp: int
    r: np.ndarray
    s: np.ndarray
    t: np.ndarray
    Dr: np.ndarray
    Ds: np.ndarray
    Dt: np.ndarray
    M: np.ndarray          # mass matrix on the reference tet (1^T M 1 = 4/3)
    Minv: np.ndarray
    LIFT: np.ndarray       # [Np, 4*Nfp], column block f is L_f = M^-1 E_f
    Fmask: np.ndarray      # [4, Nfp] element-node index of face node i of face f, ascending
    Mface: np.ndarray      # [4, Nfp, Nfp] 2-D mass matrices of the face nodes (reference triangle)
    V: np.ndarray          # Vandermonde of the (scaled) orthogonal simplex basis at the nodes
    Vinv: np.ndarray

    def interp_row(self, r0, s0, t0):
        """l_n(r0) for all n: values of the Lagrange basis at a point."""
        phi = simplex_basis(self.N, np.atleast_1d(r0), np.atleast_1d(s0), np.atleast_1d(t0))
        return (phi @ self.Vinv)[0]


def face_node_coordinates(ref_r, ref_s, ref_t, Fmask, f):
    """2-D coordinates of the nodes of face f in that face's own reference triangle."""
    idx = Fmask[f]
    if f == 0:
        return ref_r[idx], ref_s[idx]
    if f == 1:
        return ref_r[idx], ref_t[idx]
    return ref_s[idx], ref_t[idx]          # faces 2 and 3


def reference_element(N):
    assert 1 <= N <= 6
    Np, Nfp = num_nodes(N), num_face_nodes(N)
    r, s, t = warp_blend_nodes(N)
    V, Vr, Vs, Vt = simplex_basis(N, r, s, t, grad=True)
    Vinv = np.linalg.inv(V)
    Dr, Ds, Dt = Vr @ Vinv, Vs @ Vinv, Vt @ Vinv

    # mass matrix M_mn = int l_m l_n = V^-T (Gram matrix of the basis) V^-1
    qr, qs, qt, qw = tet_quadrature(N + 2)
    Phi = simplex_basis(N, qr, qs, qt)
    gram = Phi.T @ (qw[:, None] * Phi)
    M = Vinv.T @ gram @ Vinv
    M = 0.5 * (M + M.T)
    Minv = np.linalg.inv(M)

    tol = 1e-9
    face_test = (np.abs(1 + t), np.abs(1 + s), np.abs(1 + r + s + t), np.abs(1 + r))
    Fmask = np.array([np.nonzero(ft < tol)[0] for ft in face_test])
    assert Fmask.shape == (4, Nfp)

    qu, qv, qw2 = tri_quadrature(N + 2)
    Phi2 = triangle_basis(N, qu, qv)
    gram2 = Phi2.T @ (qw2[:, None] * Phi2)
    Mface = np.empty((4, Nfp, Nfp))
    LIFT = np.empty((Np, 4 * Nfp))
    for f in range(4):
        u, v = face_node_coordinates(r, s, t, Fmask, f)
        V2inv = np.linalg.inv(triangle_basis(N, u, v))
        mf = V2inv.T @ gram2 @ V2inv
        Mface[f] = 0.5 * (mf + mf.T)
        E = np.zeros((Np, Nfp))
        E[Fmask[f], :] = Mface[f]
        LIFT[:, f * Nfp:(f + 1) * Nfp] = Minv @ E
    return ReferenceElement(N=N, Np=Np, Nfp=Nfp, r=r, s=s, t=t, Dr=Dr, Ds=Ds, Dt=Dt, M=M, Minv=Minv,
                            LIFT=LIFT, Fmask=Fmask, Mface=Mface, V=V, Vinv=Vinv)
