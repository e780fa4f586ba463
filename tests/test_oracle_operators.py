"""Pins for the oracle's reference element, coefficients, geometry and connectivity (CPU only).

Every check compares the oracle with something other than itself: closed-form simplex integrals,
exact derivatives of monomials, values printed in the paper (tests/golden/), Gauss quadrature,
brute force."""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle.reference_element import (reference_element, gauss_lobatto_nodes, num_nodes,
                                      num_face_nodes, FACE_VERTICES, tri_quadrature)
from oracle.coefficients import (ab_coefficients_exact, ab_coefficients, LSERK4_A, LSERK4_B,
                                 LSERK4_C)
from oracle.mesh_geometry import (element_geometry, connect_faces, connect_faces_bruteforce,
                                  match_face_nodes, node_coordinates)
from workloads import box_tet_mesh, permute_elements

ORDERS = [1, 2, 3, 4, 5, 6]


def simplex_monomial_integral(a, b, c):
    """int over the UNIT simplex of x^a y^b z^c = a! b! c! / (a+b+c+3)!"""
    return math.factorial(a) * math.factorial(b) * math.factorial(c) / math.factorial(a + b + c + 3)


def triangle_monomial_integral(a, b):
    return math.factorial(a) * math.factorial(b) / math.factorial(a + b + 2)


@pytest.mark.parametrize("N", ORDERS)
def test_node_counts_and_faces(N, paper_coefficients):
    ref = reference_element(N)
    assert ref.Np == (N + 1) * (N + 2) * (N + 3) // 6 == num_nodes(N)
    assert ref.Fmask.shape == (4, num_face_nodes(N))
    if N == 3:
        assert ref.Np == paper_coefficients["Np_formula_check_N3"][0]
        assert paper_coefficients["unknowns_saltdome"][0] == \
            paper_coefficients["elements_saltdome"][0] * ref.Np * 4
    # face nodes really lie on their face, Fmask ascending
    r, s, t = ref.r, ref.s, ref.t
    onface = [np.abs(1 + t), np.abs(1 + s), np.abs(1 + r + s + t), np.abs(1 + r)]
    for f in range(4):
        assert np.all(onface[f][ref.Fmask[f]] < 1e-12)
        assert np.all(np.diff(ref.Fmask[f]) > 0)
        assert np.sum(onface[f] < 1e-9) == ref.Nfp


@pytest.mark.parametrize("N", ORDERS)
def test_nodes_symmetric_and_gll_on_edges(N):
    ref = reference_element(N)
    r, s, t = ref.r, ref.s, ref.t
    lam = np.stack([-(1 + r + s + t) / 2, (1 + r) / 2, (1 + s) / 2, (1 + t) / 2], axis=1)
    assert np.allclose(lam.sum(axis=1), 1.0, atol=1e-14)
    assert lam.min() > -1e-14
    for perm in itertools.permutations(range(4)):
        lp = lam[:, perm]
        d = np.abs(lp[:, None, :] - lam[None, :, :]).max(axis=2).min(axis=1)
        assert d.max() < 1e-13
    # Gauss-Lobatto points: roots of (1-x^2) P_N'(x), checked by evaluating P_N' independently
    gl = gauss_lobatto_nodes(N)
    x = gl[1:-1]
    if N >= 2:
        P = [np.ones_like(x), x]
        for n in range(1, N):
            P.append(((2 * n + 1) * x * P[n] - n * P[n - 1]) / (n + 1))
        dPN = N * (x * P[N] - P[N - 1]) / (x * x - 1)
        assert np.abs(dPN).max() < 1e-11
    for (a, b) in itertools.combinations(range(4), 2):
        on_edge = np.abs(lam[:, a] + lam[:, b] - 1) < 1e-12
        assert on_edge.sum() == N + 1
        assert np.allclose(np.sort(lam[on_edge, b] - lam[on_edge, a]), gl, atol=1e-13)


@pytest.mark.parametrize("N", ORDERS)
def test_differentiation_exact_on_polynomials(N):
    ref = reference_element(N)
    r, s, t = ref.r, ref.s, ref.t
    one = np.ones(ref.Np)
    for D in (ref.Dr, ref.Ds, ref.Dt):
        assert np.abs(D @ one).max() < 1e-12
    worst = 0.0
    for a in range(N + 1):
        for b in range(N + 1 - a):
            for c in range(N + 1 - a - b):
                f = r ** a * s ** b * t ** c
                fr = a * r ** max(a - 1, 0) * s ** b * t ** c if a else 0 * r
                fs = b * r ** a * s ** max(b - 1, 0) * t ** c if b else 0 * r
                ft = c * r ** a * s ** b * t ** max(c - 1, 0) if c else 0 * r
                worst = max(worst, np.abs(ref.Dr @ f - fr).max(), np.abs(ref.Ds @ f - fs).max(),
                            np.abs(ref.Dt @ f - ft).max())
    assert worst < 1e-12


@pytest.mark.parametrize("N", ORDERS)
def test_mass_matrix_against_closed_form_integrals(N):
    """u^T M g = int_T u g for monomials in the unit-simplex coordinates (closed form)."""
    ref = reference_element(N)
    x, y, z = (1 + ref.r) / 2, (1 + ref.s) / 2, (1 + ref.t) / 2
    assert abs(ref.M.sum() - 4.0 / 3.0) < 1e-12
    half = N // 2
    for (a, b, c) in [(0, 0, 0), (half, 0, 0), (0, half, 0), (0, 0, half), (1 if N > 1 else 0, 0, half)]:
        for (a2, b2, c2) in [(0, 0, 0), (0, N - half, 0), (N - half, 0, 0), (0, 0, N - half)]:
            if a + b + c > N or a2 + b2 + c2 > N:
                continue
            u = x ** a * y ** b * z ** c
            g = x ** a2 * y ** b2 * z ** c2
            exact = 8.0 * simplex_monomial_integral(a + a2, b + b2, c + c2)
            assert abs(u @ ref.M @ g - exact) < 1e-12


@pytest.mark.parametrize("N", ORDERS)
def test_lift_against_closed_form_face_integrals(N):
    """u^T M L_f g_f = int_face u g (reference-triangle measure, area 2) for monomials."""
    ref = reference_element(N)
    r, s, t = ref.r, ref.s, ref.t
    face_uv = [(r, s), (r, t), (s, t), (s, t)]
    for f in range(4):
        u2, v2 = face_uv[f]
        xx, yy = (1 + u2) / 2, (1 + v2) / 2           # unit-triangle coordinates on the face
        Lf = ref.LIFT[:, f * ref.Nfp:(f + 1) * ref.Nfp]
        for (a, b) in [(0, 0), (N, 0), (0, N), (N // 2, N - N // 2)]:
            for (a2, b2) in [(0, 0), (N, 0), (1, N - 1)]:
                U = xx ** a * yy ** b                  # polynomial of degree <= N in the volume
                g = (xx ** a2 * yy ** b2)[ref.Fmask[f]]
                exact = 4.0 * triangle_monomial_integral(a + a2, b + b2)
                got = U @ ref.M @ Lf @ g
                assert abs(got - exact) < 1e-11, (f, a, b, a2, b2)


def test_ab_coefficients_match_paper(paper_coefficients):
    ex = ab_coefficients_exact(3)
    g = paper_coefficients
    for s in range(3):
        assert ex["a"][s] == Fraction(*g[f"a{s + 1}"])          # eq. (18)
        assert ex["b"][s] == Fraction(*g[f"b{s + 1}"])          # eq. (19)
    for (i, j) in [(1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]:
        assert ex["C"][i - 1][j - 1] == Fraction(*g[f"C{i}{j}"])  # eq. (24)
        assert ex["C"][j - 1][i - 1] == Fraction(*g[f"C{i}{j}"])
    # reading Q1: C11 = 4703/5040 makes sum(C) = int_0^1 t^2 = 1/3; the printed value does not
    assert ex["C"][0][0] == Fraction(4703, 5040)
    assert sum(sum(row) for row in ex["C"]) == Fraction(1, 3)
    printed = Fraction(*g["C11_printed"])
    assert sum(sum(row) for row in ex["C"]) - ex["C"][0][0] + printed != Fraction(1, 3)
    assert sum(ex["abar"]) == Fraction(1, 2)


@pytest.mark.parametrize("order", [1, 2, 3])
def test_image_step_formula_against_gauss_quadrature(order):
    """Formula (24) (corrected, reading Q1) = exact integral of the product of the two AB
    interpolants (22)-(23), checked by Gauss-Legendre quadrature."""
    rng = np.random.default_rng(order)
    co = ab_coefficients(order)
    pS, pR = rng.standard_normal(2)
    rS, rR = rng.standard_normal(3), rng.standard_normal(3)
    rS[order:] = 0
    rR[order:] = 0
    dt = 0.37
    nodes = [-float(i) for i in range(order)]

    def interp(p0, rr, theta):
        # p0 + dt * int_0^theta sum_s l_s(t') r_s dt', the inner integral by quadrature as well
        xg, wg = np.polynomial.legendre.leggauss(4)
        tq = 0.5 * theta * (xg + 1)
        val = 0.0
        for s in range(order):
            ls = np.ones_like(tq)
            for j in range(order):
                if j != s:
                    ls *= (tq - nodes[j]) / (nodes[s] - nodes[j])
            val += rr[s] * np.sum(0.5 * theta * wg * ls)
        return p0 + dt * val

    xg, wg = np.polynomial.legendre.leggauss(6)
    ref_val = sum(0.5 * w * dt * interp(pS, rS, 0.5 * (x + 1)) * interp(pR, rR, 0.5 * (x + 1))
                  for x, w in zip(xg, wg))
    got = dt * (pS * pR + dt * sum(co["abar"][s] * (pS * rR[s] + pR * rS[s]) for s in range(3))
                + dt * dt * sum(co["C"][s, u] * rS[s] * rR[u] for s in range(3) for u in range(3)))
    assert abs(got - ref_val) < 1e-13 * max(1.0, abs(ref_val))
    if order == 3:
        # with the printed weights a_s instead of abar_s the formula is NOT exact (reading Q1(iii))
        wrong = dt * (pS * pR + dt * sum(co["a"][s] * (pS * rR[s] + pR * rS[s]) for s in range(3))
                      + dt * dt * sum(co["C"][s, u] * rS[s] * rR[u] for s in range(3) for u in range(3)))
        assert abs(wrong - ref_val) > 1e-3


def test_lserk4_order_conditions():
    """Butcher form of the 2N-storage scheme satisfies the eight order-4 conditions."""
    A, B, C = LSERK4_A, LSERK4_B, LSERK4_C
    s = 5
    # q_i = q_{i-1} + B_i res_i, res_i = A_i res_{i-1} + dt k_i  ->  Butcher a_ij, b_j
    coef = np.zeros((s + 1, s))      # coef[i, j]: weight of k_j in q after stage i
    res = np.zeros(s)
    for i in range(s):
        res = A[i] * res
        res[i] += 1.0
        coef[i + 1] = coef[i] + B[i] * res
    a = coef[:s]
    b = coef[s]
    c = a.sum(axis=1)
    assert np.allclose(c, C, atol=1e-14)
    conds = [(b.sum(), 1), (b @ c, 1 / 2), (b @ c ** 2, 1 / 3), (b @ a @ c, 1 / 6), (b @ c ** 3, 1 / 4),
             ((b * c) @ a @ c, 1 / 8), (b @ a @ c ** 2, 1 / 12), (b @ a @ a @ c, 1 / 24)]
    for got, want in conds:
        assert abs(got - want) < 1e-13


def test_geometry_identities():
    etov, vx = box_tet_mesh(3, 2, 2, lengths=(1.5, 1.0, 0.8), jitter=0.1, seed=7)
    geo = element_geometry(etov, vx)
    assert np.all(geo["J"] > 0)
    assert abs(geo["volume"].sum() - 1.5 * 1.0 * 0.8) < 1e-12
    closed = np.einsum("kf,kfd->kd", geo["area"], geo["normals"])
    assert np.abs(closed).max() < 1e-13                      # sum_f A_f n_f = 0
    # independent face areas / normals from cross products
    for f, fv in enumerate(FACE_VERTICES):
        p = vx[etov[:, list(fv)]]
        cr = np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0])
        assert np.allclose(0.5 * np.linalg.norm(cr, axis=1), geo["area"][:, f], rtol=1e-12)
        other = [v for v in range(4) if v not in fv][0]
        outward = np.einsum("kd,kd->k", geo["normals"][:, f], p[:, 0] - vx[etov[:, other]])
        assert np.all(outward > 0)
        assert np.allclose(np.abs(np.einsum("kd,kd->k", geo["normals"][:, f], cr))
                           , np.linalg.norm(cr, axis=1), rtol=1e-12)
    # ell = smallest height
    heights = 3.0 * geo["volume"][:, None] / geo["area"]
    assert np.allclose(geo["ell"], heights.min(axis=1))
    # chain rule (reading Q3): sum_j (d r_j/d x_i) D_j applied to the nodal coordinate x_m = delta_im
    ref = reference_element(2)
    X = node_coordinates(ref, etov, vx)
    D = (ref.Dr, ref.Ds, ref.Dt)
    for i in range(3):
        for m in range(3):
            d = sum(geo["ginv"][:, i, j, None] * (X[:, :, m] @ D[j].T) for j in range(3))
            assert np.abs(d - (1.0 if i == m else 0.0)).max() < 1e-11


def test_connectivity_bruteforce_and_counts():
    etov, vx = box_tet_mesh(3, 2, 2, jitter=0.1, seed=1)
    etov, _ = permute_elements(etov, seed=5)
    e2e, e2f = connect_faces(etov)
    b2e, b2f = connect_faces_bruteforce(etov)
    assert np.array_equal(e2e, b2e) and np.array_equal(e2f, b2f)
    # boundary triangles = 2 x boundary quads
    assert np.sum(e2e < 0) == 2 * 2 * (3 * 2 + 3 * 2 + 2 * 2)
    # symmetric
    K = etov.shape[0]
    for k in range(K):
        for f in range(4):
            if e2e[k, f] >= 0:
                assert e2e[e2e[k, f], e2f[k, f]] == k and e2f[e2e[k, f], e2f[k, f]] == f


@pytest.mark.parametrize("hexes,nb", [((4, 4, 4), 192), ((8, 8, 4), 512)])
def test_boundary_face_counts(hexes, nb):
    etov, vx = box_tet_mesh(*hexes)
    e2e, _ = connect_faces(etov)
    assert np.sum(e2e < 0) == nb         # 192 for config 1


@pytest.mark.parametrize("N", [1, 3, 4])
def test_face_node_matching_is_involution(N):
    etov, vx = box_tet_mesh(2, 2, 2, jitter=0.1, seed=3)
    ref = reference_element(N)
    e2e, e2f = connect_faces(etov)
    mapP = match_face_nodes(ref, etov, vx, e2e, e2f)
    X = node_coordinates(ref, etov, vx)
    for k in range(etov.shape[0]):
        for f in range(4):
            k2, f2 = e2e[k, f], e2f[k, f]
            if k2 < 0:
                continue
            assert np.array_equal(mapP[k2, f2][mapP[k, f]], np.arange(ref.Nfp))
            a = X[k, ref.Fmask[f]]
            b = X[k2, ref.Fmask[f2]][mapP[k, f]]
            assert np.abs(a - b).max() < 1e-12
