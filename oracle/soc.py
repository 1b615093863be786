"""Second-order cone Q_{d+1} = {(t, s) : ||s|| <= t}  --  oracle, test infrastructure.

Everything here is batched over the balls: ``a`` has shape (m,), ``B`` has shape (m, d);
row i is the point z_i = (a_i, b_i) of R^{d+1}.  The arithmetic runs in the dtype of the
inputs (float64, or float32 for the oracle's low-precision mode).
"""
from __future__ import annotations

import numpy as np

# branch codes, in the printed order of P:L115
B1 = 1  # ||b|| <= a        : Pi(z) = z
B2 = 2  # ||b|| <= -a       : Pi(z) = 0
B3 = 3  # otherwise         : Pi(z) = (a+||b||)/2 * (1, b/||b||)


def row_norms(B):
    """||b_i|| for every row, in the dtype of B."""
    return np.sqrt(np.sum(B * B, axis=1))


def branches(a, nb):
    """Branch of P:L115 for every ball, evaluated in the printed order (DESIGN reading 2)."""
    br = np.full(a.shape, B3, dtype=np.int8)
    br[nb <= -a] = B2
    br[nb <= a] = B1  # B1 is tested first in P:L115, so it wins where both hold (z = 0)
    return br


def proj_soc(a, B):
    """Pi_Q(z_i) for every ball, closed form of P:L113-115.

    Returns ``(t, PV, br, nb)`` with Pi_Q(z_i) = (t_i, PV[i, :]), the branch code and ||b_i||.
    """
    nb = row_norms(B)
    br = branches(a, nb)
    t = np.zeros_like(a)
    PV = np.zeros_like(B)
    i1 = br == B1
    t[i1] = a[i1]
    PV[i1] = B[i1]
    i3 = br == B3  # here nb > |a| >= 0, so the division is safe
    s = (a[i3] + nb[i3]) / 2
    t[i3] = s
    PV[i3] = (s / nb[i3])[:, None] * B[i3]
    return t, PV, br, nb


def dist_soc(a, B):
    """dist(z_i, Q) = ||z_i - Pi_Q(z_i)||  (definition)."""
    t, PV, _, _ = proj_soc(a, B)
    return np.sqrt((a - t) ** 2 + np.sum((B - PV) ** 2, axis=1))


def clarke_jacobian(a: float, b) -> np.ndarray:
    """One element P of the Clarke generalized Jacobian of Pi_Q at z = (a, b).

    The paper cites the formula ([7], [17]) without printing it; reading 1:
      B1 (||b|| <= a):  P = I
      B2 (||b|| <= -a): P = 0
      B3 (otherwise):   P = 1/2 [[1, w^T], [w, (1+rho) I - rho w w^T]],  w = b/||b||, rho = a/||b||
    which is the derivative of the B3 formula of P:L115 (pinned by finite differences in
    tests/test_oracle_soc.py).  On a branch boundary the predicate of P:L115 picks the element.
    """
    b = np.asarray(b, dtype=np.float64)
    d = b.shape[0]
    nb = float(np.sqrt(np.sum(b * b)))
    if nb <= a:
        return np.eye(d + 1)
    if nb <= -a:
        return np.zeros((d + 1, d + 1))
    w = b / nb
    rho = a / nb
    P = np.empty((d + 1, d + 1))
    P[0, 0] = 1.0
    P[0, 1:] = w
    P[1:, 0] = w
    P[1:, 1:] = (1.0 + rho) * np.eye(d) - rho * np.outer(w, w)
    return 0.5 * P
