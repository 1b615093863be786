"""Independent references for the MEB optimum, used only to PIN the oracle (CPU tests).

Nothing here follows ripALM: these are textbook geometry.

* ``bruteforce_meb_2d``: in the plane the minimum enclosing ball of balls is determined by a
  support set of at most 3 balls.  Enumerate every subset of 1, 2, 3 balls, build the ball
  internally tangent to the subset, and keep the smallest candidate that contains all balls.
* ``dual_lower_bound``: weak duality for problem (3) of the paper: any
  multipliers in Q^m, after being made dual feasible, give a lower bound on r*.
"""
from __future__ import annotations

import itertools
import math

import numpy as np


def _contains_all(c, r, C, R, tol):
    return bool(np.all(np.sqrt(((C - c) ** 2).sum(1)) + R <= r + tol))


def _two_ball(c1, r1, c2, r2):
    dist = math.dist(c1, c2)
    if dist + r2 <= r1 or dist + r1 <= r2:
        return None                       # one contains the other: a 1-subset candidate covers it
    r = (dist + r1 + r2) / 2
    c = c1 + (r - r1) * (c2 - c1) / dist
    return c, r


def _three_ball(c1, r1, c2, r2, c3, r3):
    """Circles internally tangent to three circles: ||c - c_i|| = r - r_i, i = 1..3."""
    A = 2 * np.array([c2 - c1, c3 - c1])
    if abs(np.linalg.det(A)) < 1e-12:
        return []
    p0 = np.array([c2 @ c2 - c1 @ c1 - (r2 * r2 - r1 * r1), c3 @ c3 - c1 @ c1 - (r3 * r3 - r1 * r1)])
    p1 = np.array([2 * (r2 - r1), 2 * (r3 - r1)])
    P = np.linalg.solve(A, p0)            # c = P + r Q
    Q = np.linalg.solve(A, p1)
    w = P - c1
    qa = Q @ Q - 1
    qb = 2 * (Q @ w + r1)
    qc = w @ w - r1 * r1
    roots = []
    if abs(qa) < 1e-14:
        if abs(qb) > 1e-14:
            roots = [-qc / qb]
    else:
        disc = qb * qb - 4 * qa * qc
        if disc >= 0:
            s = math.sqrt(disc)
            roots = [(-qb + s) / (2 * qa), (-qb - s) / (2 * qa)]
    out = []
    for r in roots:
        if r >= max(r1, r2, r3) - 1e-12:
            out.append((P + r * Q, r))
    return out


def bruteforce_meb_2d(C, R, tol=1e-9):
    C = np.asarray(C, dtype=np.float64)
    m = C.shape[0]
    assert C.shape[1] == 2
    R = np.zeros(m) if R is None else np.asarray(R, dtype=np.float64)
    best = None
    cands = [(C[i], R[i]) for i in range(m)]
    for i, j in itertools.combinations(range(m), 2):
        tb = _two_ball(C[i], R[i], C[j], R[j])
        if tb is not None:
            cands.append(tb)
    for i, j, k in itertools.combinations(range(m), 3):
        cands.extend(_three_ball(C[i], R[i], C[j], R[j], C[k], R[k]))
    for c, r in cands:
        if (best is None or r < best[1]) and _contains_all(c, r, C, R, tol * (1 + r)):
            best = (np.asarray(c, dtype=np.float64), float(r))
    return best


def dual_lower_bound(C, R, U, V):
    """Lower bound on r* from any (u_i, v_i) in Q (weak duality).

    Normalise u <- u / sum(u), v <- v / sum(u); with e = sum_i v_i set
    vt_i = (v_i - u_i e) / (1 + ||e||): then sum vt_i = 0 and ||vt_i|| <= u_i/(1+||e||)(1+||e||) ... <= u_i',
    where u_i' = u_i (the u's still sum to one).  LB = sum_i (u_i r_i + vt_i^T c_i) <= r*.
    """
    C = np.asarray(C, dtype=np.float64)
    m = C.shape[0]
    R = np.zeros(m) if R is None else np.asarray(R, dtype=np.float64)
    U = np.asarray(U, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    s = U.sum()
    u = U / s
    v = V / s
    e = v.sum(axis=0)
    ne = float(np.sqrt(e @ e))
    # (u_i, v_i - u_i e) has ||v_i - u_i e|| <= u_i (1 + ||e||); dividing BOTH by (1+||e||) keeps
    # the pair in Q but then sum u != 1; instead keep u and shrink only v: ||vt_i|| <= u_i.
    vt = (v - u[:, None] * e[None, :]) / (1.0 + ne)
    assert np.all(np.sqrt((vt ** 2).sum(1)) <= u * (1 + 1e-12) + 1e-300)
    assert np.abs(vt.sum(axis=0)).max() <= 1e-12
    return float(u @ R + np.sum(vt * C))
