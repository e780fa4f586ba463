"""ORACLE (test infrastructure) - time-integration coefficients by exact rational integration.

Adams-Bashforth of order m = 1,2,3 interpolates the right-hand side through the local steps
0, -1, .., -(m-1) (unit = the local time step) with Lagrange functions l_s, s = 1..m
(PAPER.md:182-188).  With I_s(theta) = int_0^theta l_s:
    a_s    = I_s(1)                    update weights, eq. (18)
    b_s    = I_s(1/2)                  half-step weights, eq. (19)
    abar_s = int_0^1 I_s               first-order image weights   (reading Q1(iii))
    C_st   = int_0^1 I_s I_t           second-order image weights, matrix C of eq. (24)
The paper prints a_s in lines 2-3 of (24) and C_11 = 4703/50400; exact integration gives abar_s and
C_11 = 4703/5040 (reading Q1), which is what is returned here.
Orders 1 and 2 are used during start-up (reading Q7).

LSERK4: the five-stage fourth-order 2N-storage Runge-Kutta scheme of Carpenter & Kennedy (1994),
needed only by BASELINE.json config 1 (not in the paper, reading Q8).
"""
from fractions import Fraction
from functools import lru_cache

import numpy as np


def _poly_mul(p, q):
    out = [Fraction(0)] * (len(p) + len(q) - 1)
    for i, a in enumerate(p):
        for j, b in enumerate(q):
            out[i + j] += a * b
    return out


def _poly_int(p):
    """Antiderivative vanishing at 0 (coefficients ascending)."""
    return [Fraction(0)] + [c / (i + 1) for i, c in enumerate(p)]


def _poly_eval(p, x):
    return sum(c * x ** i for i, c in enumerate(p))


def lagrange_on_past_steps(order):
    """l_s(t), s = 1..order, through the nodes 0, -1, .., -(order-1); ascending coefficients."""
    nodes = [Fraction(-i) for i in range(order)]
    polys = []
    for s in range(order):
        p = [Fraction(1)]
        for j in range(order):
            if j != s:
                p = _poly_mul(p, [-nodes[j] / (nodes[s] - nodes[j]), 1 / (nodes[s] - nodes[j])])
        polys.append(p)
    return polys


def ab_coefficients_exact(order):
    """dict of Fractions: a[s], b[s], abar[s], C[s][t] (lists of length `order`)."""
    I = [_poly_int(p) for p in lagrange_on_past_steps(order)]
    one, half = Fraction(1), Fraction(1, 2)
    a = [_poly_eval(p, one) for p in I]
    b = [_poly_eval(p, half) for p in I]
    abar = [_poly_eval(_poly_int(p), one) for p in I]
    C = [[_poly_eval(_poly_int(_poly_mul(p, q)), one) for q in I] for p in I]
    return dict(a=a, b=b, abar=abar, C=C)


@lru_cache(maxsize=None)
def ab_coefficients(order):
    """Same as floats, zero-padded to three history slots: a[3], b[3], abar[3], C[3,3]."""
    ex = ab_coefficients_exact(order)
    out = dict(a=np.zeros(3), b=np.zeros(3), abar=np.zeros(3), C=np.zeros((3, 3)))
    for s in range(order):
        out["a"][s] = float(ex["a"][s])
        out["b"][s] = float(ex["b"][s])
        out["abar"][s] = float(ex["abar"][s])
        for t in range(order):
            out["C"][s, t] = float(ex["C"][s][t])
    return out


# Carpenter-Kennedy low-storage RK4(5) coefficients (literature values; reading Q8)
LSERK4_A = np.array([0.0,
                     -567301805773.0 / 1357537059087.0,
                     -2404267990393.0 / 2016746695238.0,
                     -3550918686646.0 / 2091501179385.0,
                     -1275806237668.0 / 842570457699.0])
LSERK4_B = np.array([1432997174477.0 / 9575080441755.0,
                     5161836677717.0 / 13612068292357.0,
                     1720146321549.0 / 2090206949498.0,
                     3134564353537.0 / 4481467310338.0,
                     2277821191437.0 / 14882151754819.0])
LSERK4_C = np.array([0.0,
                     1432997174477.0 / 9575080441755.0,
                     2526269341429.0 / 6820363962896.0,
                     2006345519317.0 / 3224310063776.0,
                     2802321613138.0 / 2924317926251.0])
