"""ripALM for the minimum enclosing ball of balls  --  oracle drivers, test infrastructure.

Follows the paper step by step, in its order and notation:

* ``ssn``       Algorithm 2: semismooth Newton for the subproblem (4).
* ``ripalm``    Algorithm 1: outer loop, multiplier update (6), auxiliary
                sequence (alpha, beta), stopping by KKT_max.
* ``meb_solve`` the whole solve, FP64 mode or the mixed-precision reduction of
                Section 4.2.

Where the paper is silent the readings of DESIGN.md ("Readings of the paper", same numbers
as SURVEY.md §8(c)) are taken; each place is marked ``[reading n]``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import primitives as prim
from . import soc


@dataclass
class Params:
    """Free constants of Algorithms 1-2 and Section 4.2.

    The paper lists them as inputs without values; [reading 3, 4, 5, 9, 10, 12].
    """
    rho: float = 0.5              # rho in [0,1) of condition (5)
    sigma0: float = 1.0           # sigma_0 (normalised units)
    kappa: float = 3.0            # sigma_{k+1} = min(sigma_max, kappa sigma_k)
    sigma_max: float = 1e8
    tau: float = 1.0              # tau_k constant (satisfies P:L155 with nu_k = 0)
    armijo_mu: float = 1e-4       # "standard Armijo line search"
    armijo_max_halvings: int = 30
    cg_max: int = 500             # matrix-free Krylov solve
    dense_d_max: int = 128        # "moderate d": dense factorisation for d <= this
    inner_max: int = 50
    outer_max: int = 200
    tol_lo: float = 1e-2          # low-precision stopping tolerance
    tol_red_factor: float = 0.02  # tol_red = 0.02 r_hat  [reading 9], pinned by Table 1
    max_rounds: int = 10          # active-set refinement rounds
    sample_rows: int = 1024       # rows whose mean is the initial centre c^0
    ag_outer: int = 0             # outer iterations k < ag_outer use the accelerated gradient inner solver
    ag_inner_max: int = 500       # its iteration cap  [reading 20]


@dataclass
class Stats:
    outer: int = 0
    newton: int = 0
    evals: int = 0          # evaluations of the ALM map over the balls (= passes)
    cg_iters: int = 0
    kkt: float = np.inf
    kkt_terms: tuple = ()
    converged: bool = False
    history: list = field(default_factory=list)


def rel_kkt(ev, r_norm, length_unit):
    """Maximum KKT residual on the tentative multipliers of ``ev``.

    [reading 7] "1e-8 relative KKT": the two length-valued terms (primal cone distance and
    complementarity) are divided by (1 + r) with r in the units of the raw data;
    ``length_unit`` = L converts the normalised lengths back (raw = L * normalised).
    """
    Lr = length_unit
    g0 = abs(1.0 - ev["sum_uplus"])                        # |1 - sum u_i|
    g1 = float(np.sqrt(np.sum(ev["sum_vplus"] ** 2)))      # ||sum v_i||
    denom = 1.0 + Lr * r_norm
    p = Lr * ev["max_pfeas"] / denom
    dd = ev["max_dfeas"]
    cp = Lr * ev["max_compl"] / denom
    terms = (g0, g1, p, dd, cp)
    return max(terms), terms


def condition5(ev, x, xbar, alphabeta, sigma, tau, rho):
    """Relative-type stopping condition (5), on the tentative quantities."""
    g = ev["grad"]
    lhs = 2.0 * sigma * abs(float((alphabeta - x) @ g)) + sigma ** 2 * float(g @ g)
    dx = x - xbar
    rhs = rho * (ev["sum_dmult2"] + tau * float(dx @ dx))
    return lhs <= rhs


def newton_direction(C, R, U, V, x, sigma, tau, g, par: Params, dtype, stats: Stats):
    """Solve H Delta = -g.  Dense factorisation for moderate d,
    matrix-free CG otherwise [reading 5]."""
    d = C.shape[1]
    if d <= par.dense_d_max:
        H, _ = prim.dense_hessian(C, R, U, V, x, sigma, tau, dtype)
        Lc = np.linalg.cholesky(H)                     # H is SPD
        y = np.linalg.solve(Lc, -g)
        return np.linalg.solve(Lc.T, y)
    # conjugate gradients on H Delta = -g, stop ||H Delta + g|| <= min(0.1, ||g||) ||g||
    gn = float(np.sqrt(g @ g))
    tol = min(0.1, gn) * gn
    delta = np.zeros_like(g)
    res = -g.copy()            # residual of H delta = -g at delta = 0
    p = res.copy()
    rr = float(res @ res)
    for _ in range(par.cg_max):
        if np.sqrt(rr) <= tol:
            break
        Hp, _ = prim.hvp(C, R, U, V, x, sigma, tau, p, dtype)
        stats.cg_iters += 1
        alpha = rr / float(p @ Hp)
        delta += alpha * p
        res -= alpha * Hp
        rr_new = float(res @ res)
        p = res + (rr_new / rr) * p
        rr = rr_new
    return delta


def ssn(C, R, U, V, x, xbar, alphabeta, sigma, tau, tol, par: Params, dtype, length_unit,
        stats: Stats):
    """Algorithm 2.  Returns ``(x, ev, status)``; ``ev`` is the evaluation at the
    returned x, holding the tentative multipliers."""
    ev = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau, dtype)          # lines 3-4
    stats.evals += 1
    status = "cap"
    for _ in range(par.inner_max):
        kkt, _ = rel_kkt(ev, x[0], length_unit)
        if condition5(ev, x, xbar, alphabeta, sigma, tau, par.rho):     # line 5
            status = "cond5"
            break
        if kkt <= tol:                                                  # [reading 6]
            status = "kkt"
            break
        g = ev["grad"]
        delta = newton_direction(C, R, U, V, x, sigma, tau, g, par, dtype, stats)  # line 8
        stats.newton += 1
        # Armijo line search for Psi [reading 4]
        slope = float(g @ delta)
        eta = 1.0
        accepted = False
        ev_t = None
        for _ls in range(par.armijo_max_halvings + 1):
            x_t = x + eta * delta
            ev_t = prim.eval_alm(C, R, U, V, x_t, xbar, sigma, tau, dtype)
            stats.evals += 1
            if ev_t["psi_var"] <= ev["psi_var"] + par.armijo_mu * eta * slope:
                accepted = True
                break
            eta *= 0.5
        if not accepted:
            if ev_t["psi_var"] <= ev["psi_var"]:
                x, ev = x_t, ev_t       # last trial did not increase Psi: take it
            status = "stalled"
            break
        x, ev = x_t, ev_t               # the accepted trial is the next iteration's evaluation
    return x, ev, status


def accelerated_gradient(C, R, U, V, x, xbar, alphabeta, sigma, tau, tol, par: Params, dtype, length_unit,
                         stats: Stats):
    """Accelerated gradient method for the subproblem (4)  ("First-order methods, including accelerated
    gradient methods [4], provide simple inner solvers ... attractive in the early outer iterations").
    [reading 20] FISTA with backtracking on the Lipschitz estimate and the gradient restart:
        x+ = y - grad Psi(y) / Lip,  accepted when Psi(x+) <= Psi(y) - ||grad Psi(y)||^2 / (2 Lip), else Lip <- 2 Lip;
        t+ = (1 + sqrt(1 + 4 t^2)) / 2,   y+ = x+ + ((t - 1) / t+) (x+ - x);   restart (t = 1, y+ = x+) when
        <grad Psi(y), x+ - x> > 0.
    Lip starts at tau/sigma + sigma * (number of active balls at x), the norm bound of H there (||P_i|| <= 1).
    Same stopping tests as Algorithm 2 (condition (5) or KKT_max on the tentative quantities).  Returns (x, ev, status)."""
    ev = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau, dtype)
    stats.evals += 1
    status = "cap"
    y = x.copy()
    ev_y = ev
    t = 1.0
    lip = tau / sigma + sigma * max(1, ev["n_b1"] + ev["n_b3"])
    for _ in range(par.ag_inner_max):
        kkt, _ = rel_kkt(ev, x[0], length_unit)
        if condition5(ev, x, xbar, alphabeta, sigma, tau, par.rho):
            status = "cond5"
            break
        if kkt <= tol:
            status = "kkt"
            break
        g_y = ev_y["grad"]
        gg = float(g_y @ g_y)
        accepted = False
        for _bt in range(60):
            x_new = y - g_y / lip
            ev_new = prim.eval_alm(C, R, U, V, x_new, xbar, sigma, tau, dtype)
            stats.evals += 1
            if ev_new["psi_var"] <= ev_y["psi_var"] - 0.5 * gg / lip:
                accepted = True
                break
            lip *= 2.0
        if not accepted:
            status = "stalled"
            break
        restart = float(g_y @ (x_new - x)) > 0.0
        t_new = 1.0 if restart else 0.5 * (1.0 + np.sqrt(1.0 + 4.0 * t * t))
        y = x_new.copy() if restart else x_new + ((t - 1.0) / t_new) * (x_new - x)
        x, ev, t = x_new, ev_new, t_new
        if np.array_equal(y, x):
            ev_y = ev                      # the evaluation at x+ is the evaluation at y
        else:
            ev_y = prim.eval_alm(C, R, U, V, y, xbar, sigma, tau, dtype)
            stats.evals += 1
    return x, ev, status


def ripalm(C, R, x0, alphabeta0, U0, V0, tol, par: Params, dtype=np.float64, length_unit=1.0,
           sigma0=None):
    """Algorithm 1 on the data as given.  Terminates when the maximum KKT
    residual is below ``tol``.  Returns ``(x, U, V, stats)``."""
    st = Stats()
    x = np.asarray(x0, dtype=np.float64).copy()
    ab = np.asarray(alphabeta0, dtype=np.float64).copy()
    U = np.asarray(U0, dtype=dtype).copy()
    V = np.asarray(V0, dtype=dtype).copy()
    sigma = par.sigma0 if sigma0 is None else sigma0
    tau = par.tau
    for k in range(par.outer_max):
        xbar = x.copy()                                                   # (r^k, c^k)
        inner = accelerated_gradient if k < par.ag_outer else ssn         # P:L204 / Algorithm 2
        x, ev, status = inner(C, R, U, V, x, xbar, ab, sigma, tau, tol, par, dtype,
                              length_unit, st)                            # step 3
        U = ev["Uplus"].copy()                                            # eq. (6)
        V = ev["Vplus"].copy()
        ab = ab - sigma * ev["grad"]                                      # step 4
        st.outer = k + 1
        st.kkt, st.kkt_terms = rel_kkt(ev, x[0], length_unit)
        st.history.append((k, sigma, status, st.kkt, st.evals, ev["n_b1"], ev["n_b3"]))
        if st.kkt <= tol:
            st.converged = True
            break
        sigma = min(par.sigma_max, par.kappa * sigma)                     # P:L175 [reading 3]
    return x, U, V, st


# ------------------------------------------------------------------------------------
def initial_point(C, R, par: Params):
    """[reading 3] c^0 = mean of a fixed strided sample of the centres (rows floor(k m / S),
    S = min(m, sample_rows)); r^0 = L = max_i (||c_i - c^0|| + r_i), so x^0 is feasible."""
    m = C.shape[0]
    S = min(m, par.sample_rows)
    rows = (np.arange(S, dtype=np.int64) * m) // S
    c0 = C[rows].mean(axis=0)
    Rr = np.zeros(m) if R is None else R
    L = float(np.max(soc.row_norms(C - c0[None, :]) + Rr))
    return c0, L


def meb_solve(C, R, tol=1e-8, mode="fp64", par: Params | None = None):
    """Minimum enclosing ball of the balls (c_i, r_i)  (MEB).

    mode "fp64":  Algorithm 1 in float64 on all m balls.
    mode "mixed": Section 4.2: float32 run to ``tol_lo`` on all m, boundary
                  screening, float64 run on the reduced problem warm-started
                  from the coarse solution, full float64 feasibility check and
                  re-introduction of violated balls.

    Returns ``(center, radius, info)``.  The returned radius is
    r_out = max_i (||c - c_i|| + r_i) for the returned centre  [reading 10 / step 7].
    """
    par = Params() if par is None else par
    C = np.asarray(C, dtype=np.float64)
    m, d = C.shape
    Rz = np.zeros(m) if R is None else np.asarray(R, dtype=np.float64)
    c0, L = initial_point(C, R, par)
    info = dict(mode=mode, m=m, d=d, L=L, phases=[], n_red=[], rounds=0)
    if L == 0.0:                                      # [reading 16] all balls are the point c0
        info.update(converged=True, delta_max=0.0)
        return c0, 0.0, info
    # [reading 3] the algorithm runs on the normalised instance (c_i - c^0)/L, r_i/L
    Cn = (C - c0[None, :]) / L
    Rn = Rz / L
    x0 = np.zeros(d + 1)
    x0[0] = 1.0

    if mode == "fp64":
        x, U, V, st = ripalm(Cn, Rn, x0, x0, np.zeros(m), np.zeros((m, d)), tol, par,
                             np.float64, L)
        info["phases"].append(("fp64-full", m, st))
        converged = st.converged
    elif mode == "mixed":
        # phase 1: low precision, loose tolerance, all m  [reading 8]
        C32 = Cn.astype(np.float32)
        R32 = Rn.astype(np.float32)
        x, U32, V32, st1 = ripalm(C32, R32, x0, x0, np.zeros(m, np.float32),
                                  np.zeros((m, d), np.float32), par.tol_lo, par, np.float32, L)
        info["phases"].append(("fp32-full", m, st1))
        # screening, in float32, tol_red = 0.02 r_hat  [reading 9]
        tol_red = par.tol_red_factor * x[0]
        flags, _ = prim.screen_flags(C32, R32, x[0], x[1:], tol_red)
        I = prim.compact(flags)
        if I.size == 0:   # cannot happen for a sensible r_hat; keep the farthest ball at least
            I = np.array([int(np.argmax(soc.row_norms(Cn - x[1:][None, :]) + Rn))], np.int32)
        U = U32[I].astype(np.float64)                  # warm start restricted to I_red
        V = V32[I].astype(np.float64)
        ab = x.copy()                                  # [reading 11]
        converged = False
        for rnd in range(par.max_rounds):
            info["n_red"].append(int(I.size))
            x, U, V, st2 = ripalm(Cn[I], Rn[I], x, ab, U, V, tol, par, np.float64, L)
            info["phases"].append(("fp64-reduced", int(I.size), st2))
            info["rounds"] = rnd + 1
            # a-posteriori check against ALL original constraints, raw data
            r_raw = L * x[0]
            c_raw = c0 + L * x[1:]
            eps_feas = tol * (1.0 + r_raw)             # [reading 10]
            kept = np.zeros(m, dtype=bool)
            kept[I] = True
            dmax, _, viol_idx, _ = prim.feasibility_check(C, R, r_raw, c_raw, eps_feas, kept)
            if viol_idx.size == 0:
                converged = st2.converged
                break
            # re-introduce the violated balls with zero multipliers [reading 12]
            I = np.concatenate([I, viol_idx])
            U = np.concatenate([U, np.zeros(viol_idx.size)])
            V = np.concatenate([V, np.zeros((viol_idx.size, d))])
            ab = x.copy()
    else:
        raise ValueError(mode)

    c_out = c0 + L * x[1:]
    r_out, amax, _, _ = prim.feasibility_check(C, R, 0.0, c_out, np.inf)   # max_i(||c-c_i|| + r_i)
    info.update(converged=bool(converged), r_alg=L * x[0], argmax=amax,
                delta_max=r_out - L * x[0], x_norm=x, U=U, V=V,
                index_set=(None if mode == "fp64" else I), c0=c0)
    return c_out, float(r_out), info
