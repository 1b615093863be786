"""Per-primitive oracle: one plain pass over the balls each  --  test infrastructure.

Layout is the paper's structure-of-arrays: R (m,), C (m, d), U (m,), V (m, d)
(V is DENSE here; the CUDA path stores only the rows with u_i > 0, which is the same
mathematical object because u_i = 0 implies v_i = 0 for multipliers in Q).

Notation:  z_i = (a_i, b_i),  a_i = r_i - r + u_i/sigma,
b_i = c_i - c + v_i/sigma,  x = (r, c),  xbar = (rbar, cbar) the proximal centre.

``dtype=np.float32`` is the oracle's low-precision mode (DESIGN reading 8): the data and
the per-ball arithmetic are float32, every sum over balls and the (d+1)-state are float64.

Sums over the balls are accumulated more accurately than float64 recursive summation
(math.fsum for scalars, long double / pairwise for vectors) so that the oracle is the more
accurate side of a parity comparison.  Each reduction also returns the sum of absolute
values of its terms ("scale"), which is the denominator of the relative parity error
(DESIGN.md "Parity metrics").
"""
from __future__ import annotations

import math

import numpy as np

from . import soc


# ----------------------------------------------------------------------------- sums
def _ssum(x) -> float:
    """Exactly rounded sum of a 1-D array (float64 result)."""
    return math.fsum(np.asarray(x, dtype=np.float64).tolist())


def _colsum(X) -> np.ndarray:
    """Column sums of an (m, d) array, accumulated in long double (or pairwise if huge)."""
    X = np.asarray(X)
    if X.shape[0] == 0:
        return np.zeros(X.shape[1])
    if X.size <= 2_000_000:
        return X.T.astype(np.longdouble).sum(axis=1).astype(np.float64)
    return np.sum(np.ascontiguousarray(X.T, dtype=np.float64), axis=1)  # pairwise along rows


# ----------------------------------------------------------------------------- z_i
def shifted_points(C, R, U, V, x, sigma, dtype=np.float64):
    """a_i, b_i of P:L191 / P:L228 in ``dtype``.  R None means points (r_i = 0)."""
    dt = np.dtype(dtype).type
    C = np.asarray(C, dtype=dtype)
    m = C.shape[0]
    Rr = np.zeros(m, dtype=dtype) if R is None else np.asarray(R, dtype=dtype)
    Uu = np.asarray(U, dtype=dtype)
    Vv = np.asarray(V, dtype=dtype)
    r = dt(x[0])
    c = np.asarray(x[1:], dtype=dtype)
    sg = dt(sigma)
    a = Rr - r + Uu / sg
    B = C - c[None, :] + Vv / sg
    return a, B, Rr, C, Uu, Vv, r, c, sg


# ----------------------------------------------------------------------------- a1
def eval_alm(C, R, U, V, x, xbar, sigma, tau, dtype=np.float64):
    """One evaluation of the proximal augmented Lagrangian at x.

    P:L107 (phi_sigma), P:L111 (gradient), P:L131 (Psi_k), P:L139 (tentative multipliers),
    P:L187 / P:L232 (g), right side of (5) P:L135, KKT terms P:L309.

    Returns a dict:
      psi_var     r + (sigma/2) sum ||Pi(z_i)||^2 + (tau/2sigma) ||x - xbar||^2
                  (Psi without the term that is constant in x, DESIGN reading 13)
      grad        (1;0) - (sum u+; sum v+) + (tau/sigma)(x - xbar)            (d+1,)
      sum_uplus, sum_vplus, sum_proj2, sum_dmult2, n_b1, n_b3
      max_pfeas   max_i dist((r - r_i, c - c_i), Q)
      max_dfeas   max_i dist((u+_i, v+_i), Q)
      max_compl   max_i |(r - r_i) u+_i + <c - c_i, v+_i>|
      per-ball:   a, nb, br, t, lam (Pi(z_i) = (t_i, lam_i b_i)), Uplus, Vplus
      scales:     scale_* = sum of |terms| of the reduction of the same name
    """
    x = np.asarray(x, dtype=np.float64)
    xbar = np.asarray(xbar, dtype=np.float64)
    a, B, Rr, Cc, Uu, Vv, r, c, sg = shifted_points(C, R, U, V, x, sigma, dtype)
    t, PV, br, nb = soc.proj_soc(a, B)
    Uplus = sg * t                                           # P:L139 / P:L183
    Vplus = sg * PV
    proj2 = t * t + np.sum(PV * PV, axis=1)                  # ||Pi(z_i)||^2
    dmult2 = (Uplus - Uu) ** 2 + np.sum((Vplus - Vv) ** 2, axis=1)   # right side of (5)
    pfeas = soc.dist_soc(r - Rr, c[None, :] - Cc)            # P:L309 third term
    dfeas = soc.dist_soc(Uplus, Vplus)                       # P:L309 fourth term
    compl = np.abs((r - Rr) * Uplus + np.sum((c[None, :] - Cc) * Vplus, axis=1))  # fifth term

    # lam_i with Pi(z_i) = (t_i, lam_i b_i): 1 on B1, 0 on B2, s/nb on B3
    lam = np.zeros_like(a)
    lam[br == soc.B1] = 1
    i3 = br == soc.B3
    lam[i3] = t[i3] / nb[i3]

    sum_uplus = _ssum(Uplus)
    sum_vplus = _colsum(Vplus)
    sum_proj2 = _ssum(proj2)
    sum_dmult2 = _ssum(dmult2)
    sigma = float(sigma)
    tau = float(tau)
    dx = x - xbar
    psi_var = float(x[0]) + 0.5 * sigma * sum_proj2 + 0.5 * (tau / sigma) * float(dx @ dx)
    grad = np.zeros_like(x)
    grad[0] = 1.0
    grad[0] -= sum_uplus
    grad[1:] -= sum_vplus
    grad += (tau / sigma) * dx                               # P:L187 / P:L232
    m = a.shape[0]
    return dict(
        psi_var=psi_var, grad=grad,
        sum_uplus=sum_uplus, sum_vplus=sum_vplus, sum_proj2=sum_proj2, sum_dmult2=sum_dmult2,
        n_b1=int(np.count_nonzero(br == soc.B1)), n_b3=int(np.count_nonzero(i3)),
        max_pfeas=float(pfeas.max()) if m else 0.0,
        max_dfeas=float(dfeas.max()) if m else 0.0,
        max_compl=float(compl.max()) if m else 0.0,
        a=a, nb=nb, br=br, t=t, lam=lam, Uplus=Uplus, Vplus=Vplus,
        pfeas=pfeas, compl=compl,
        scale_uplus=_ssum(np.abs(Uplus)),
        scale_vplus=_colsum(np.abs(Vplus)),
        scale_proj2=sum_proj2,
        scale_dmult2=_ssum(Uplus.astype(np.float64) ** 2 + Uu.astype(np.float64) ** 2
                           + np.sum(Vplus.astype(np.float64) ** 2, axis=1)
                           + np.sum(Vv.astype(np.float64) ** 2, axis=1)),
    )


# ----------------------------------------------------------------------------- a2
def hvp(C, R, U, V, x, sigma, tau, q, dtype=np.float64):
    """H q = (tau/sigma) q + sigma sum_i P_i q   (P_i: DESIGN reading 1).

    Returns ``(Hq, scale)``, scale = (tau/sigma)|q| + sigma sum_i |P_i q| componentwise.
    """
    x = np.asarray(x, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    a, B, *_ = shifted_points(C, R, U, V, x, sigma, dtype)
    dt = np.dtype(dtype).type
    nb = soc.row_norms(B)
    br = soc.branches(a, nb)
    q0 = dt(q[0])
    q1 = np.asarray(q[1:], dtype=dtype)
    m, d = B.shape
    P0 = np.zeros(m, dtype=dtype)       # (P_i q)_0
    P1 = np.zeros((m, d), dtype=dtype)  # (P_i q)_1
    i1 = br == soc.B1                   # P_i = I
    P0[i1] = q0
    P1[i1] = q1[None, :]
    i3 = br == soc.B3                   # P_i = 1/2 [[1, w^T], [w, (1+rho) I - rho w w^T]]
    W = B[i3] / nb[i3][:, None]
    rho = a[i3] / nb[i3]
    wq = W @ q1
    P0[i3] = (q0 + wq) / 2
    P1[i3] = (q0 * W + (1 + rho)[:, None] * q1[None, :] - (rho * wq)[:, None] * W) / 2
    sigma = float(sigma)
    tau = float(tau)
    S = np.concatenate([[_ssum(P0)], _colsum(P1)])
    Sabs = np.concatenate([[_ssum(np.abs(P0))], _colsum(np.abs(P1))])
    Hq = (tau / sigma) * q + sigma * S
    scale = (tau / sigma) * np.abs(q) + sigma * Sabs
    return Hq, scale


# ----------------------------------------------------------------------------- a2'
def dense_hessian_loop(C, R, U, V, x, sigma, tau):
    """H = (tau/sigma) I + sigma sum_i P_i, summing explicit matrices ball by ball.

    Pure-Python loop: small cases only.  This is the definition the vectorised
    ``dense_hessian`` is pinned against.
    """
    x = np.asarray(x, dtype=np.float64)
    a, B, *_ = shifted_points(C, R, U, V, x, sigma)
    d = B.shape[1]
    S = np.zeros((d + 1, d + 1))
    for i in range(B.shape[0]):
        S += soc.clarke_jacobian(float(a[i]), B[i])
    return (float(tau) / float(sigma)) * np.eye(d + 1) + float(sigma) * S


def dense_hessian(C, R, U, V, x, sigma, tau, dtype=np.float64):
    """Same matrix as ``dense_hessian_loop`` written with sums over the B3 balls
    (SURVEY §8(a) row a2'):  sum_i P_i = n1 I + 1/2 [[n3, s^T], [s, (n3 + sum rho) I - W^T diag(rho) W]],
    s = sum_i w_i.  Returns ``(H, scale)`` with scale the matrix of sums of |terms|."""
    x = np.asarray(x, dtype=np.float64)
    a, B, *_ = shifted_points(C, R, U, V, x, sigma, dtype)
    nb = soc.row_norms(B)
    br = soc.branches(a, nb)
    d = B.shape[1]
    n1 = int(np.count_nonzero(br == soc.B1))
    i3 = br == soc.B3
    n3 = int(np.count_nonzero(i3))
    W = (B[i3] / nb[i3][:, None]).astype(np.float64)
    rho = (a[i3] / nb[i3]).astype(np.float64)
    S = np.zeros((d + 1, d + 1))
    S[0, 0] = n3
    s = _colsum(W)
    S[0, 1:] = s
    S[1:, 0] = s
    S[1:, 1:] = (n3 + _ssum(rho)) * np.eye(d) - (W.T * rho[None, :]) @ W
    sigma = float(sigma)
    tau = float(tau)
    H = (tau / sigma) * np.eye(d + 1) + sigma * (n1 * np.eye(d + 1) + 0.5 * S)
    A = np.zeros((d + 1, d + 1))
    A[0, 0] = n3
    sa = _colsum(np.abs(W))
    A[0, 1:] = sa
    A[1:, 0] = sa
    A[1:, 1:] = (n3 + _ssum(np.abs(rho))) * np.eye(d) + (np.abs(W).T * np.abs(rho)[None, :]) @ np.abs(W)
    scale = (tau / sigma) * np.eye(d + 1) + sigma * (n1 * np.eye(d + 1) + 0.5 * A)
    return H, scale


# ----------------------------------------------------------------------------- a6
def update_multipliers(C, R, U, V, x, sigma, dtype=np.float64):
    """(u_i, v_i)^+ = sigma Pi_Q(z_i) for all i  (eq. (6); batched form P:L181-183).

    Returns ``(Uplus, Vplus, sum_mult2)`` with sum_mult2 = sum_i (u+_i^2 + ||v+_i||^2)
    (the sum in the last term of phi_sigma)."""
    x = np.asarray(x, dtype=np.float64)
    a, B, *_rest, sg = shifted_points(C, R, U, V, x, sigma, dtype)
    t, PV, _, _ = soc.proj_soc(a, B)
    Uplus = sg * t
    Vplus = sg * PV
    m2 = Uplus.astype(np.float64) ** 2 + np.sum(Vplus.astype(np.float64) ** 2, axis=1)
    return Uplus, Vplus, _ssum(m2)


# ----------------------------------------------------------------------------- a7
def screen_slack(C32, R32, r_hat, c_hat):
    """Approximate slack s_i = r_hat - r_i - ||c_hat - c_i|| in float32."""
    C32 = np.asarray(C32, dtype=np.float32)
    m = C32.shape[0]
    R32 = np.zeros(m, dtype=np.float32) if R32 is None else np.asarray(R32, dtype=np.float32)
    ch = np.asarray(c_hat, dtype=np.float32)
    dist = soc.row_norms(ch[None, :] - C32)
    return np.float32(r_hat) - R32 - dist


def screen_flags(C32, R32, r_hat, c_hat, tol_red):
    """Retain rule I_red = {i : s_i <= tol_red}.  Returns (flags uint8, slack)."""
    s = screen_slack(C32, R32, r_hat, c_hat)
    return (s <= np.float32(tol_red)).astype(np.uint8), s


def compact(flags):
    """Ascending int32 index list of the set flags (stream compaction = flatnonzero)."""
    return np.flatnonzero(np.asarray(flags)).astype(np.int32)


# ----------------------------------------------------------------------------- a8
def feasibility_check(C, R, r, c, eps_feas, kept_mask=None):
    """Delta_max = max_i (r_i + ||cbar - c_i|| - rbar) over ALL balls, its argmax (smallest
    index on ties) and the violated set V = {i not kept : viol_i > eps_feas}.

    Returns ``(delta_max, argmax, viol_idx int32 ascending, viol)``."""
    C = np.asarray(C, dtype=np.float64)
    m = C.shape[0]
    Rr = np.zeros(m) if R is None else np.asarray(R, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    viol = Rr + soc.row_norms(c[None, :] - C) - float(r)
    amax = int(np.argmax(viol))  # first occurrence = smallest index on ties
    bad = viol > float(eps_feas)
    if kept_mask is not None:
        bad &= ~(np.asarray(kept_mask).astype(bool))
    return float(viol[amax]), amax, np.flatnonzero(bad).astype(np.int32), viol


# ----------------------------------------------------------------------------- a1 along a line
def eval_alm_line(C, R, U, V, x, xbar, sigma, tau, direction, gammas, dtype=np.float64):
    """psi_var at the points x - gamma * direction, one plain evaluation per gamma (the definition the CUDA
    path's single-pass multi-trial evaluation is compared with).  Returns a list of
    ``(psi_var, psi_scale)`` with psi_scale = |r| + (sigma/2) sum ||Pi(z_i)||^2 + (tau/2sigma)||x - xbar||^2."""
    x = np.asarray(x, dtype=np.float64)
    direction = np.asarray(direction, dtype=np.float64)
    out = []
    for g in gammas:
        xg = x - float(g) * direction
        ev = eval_alm(C, R, U, V, xg, xbar, sigma, tau, dtype)
        dx = xg - np.asarray(xbar, dtype=np.float64)
        scale = abs(xg[0]) + 0.5 * float(sigma) * ev["scale_proj2"] + 0.5 * (float(tau) / float(sigma)) * float(dx @ dx)
        out.append((ev["psi_var"], scale))
    return out
