"""Pins for oracle/ripalm.py (CPU only): the solver's answer against closed forms, brute force
in the plane, a primal-dual certificate, KKT invariants and the paper's Table 1."""
import os

import numpy as np
import pytest

import workloads
from oracle import primitives as prim
from oracle import ripalm
from tests._meb_reference_forms import bruteforce_meb_2d, dual_lower_bound

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
MODES = ["fp64", "mixed"]


@pytest.mark.parametrize("mode", MODES)
def test_two_balls_closed_form(mode):
    # r = (||c1 - c2|| + r1 + r2)/2, centre on the segment at distance r - r1 from c1
    c1, r1 = np.array([1.0, 2.0, -1.0, 0.5]), 0.7
    c2, r2 = np.array([-2.0, 0.0, 3.0, 1.5]), 1.9
    dist = np.linalg.norm(c1 - c2)
    r_want = (dist + r1 + r2) / 2
    c_want = c1 + (r_want - r1) * (c2 - c1) / dist
    c, r, info = ripalm.meb_solve(np.array([c1, c2]), np.array([r1, r2]), 1e-10, mode)
    assert info["converged"]
    assert abs(r - r_want) <= 1e-9 * r_want
    np.testing.assert_allclose(c, c_want, atol=1e-8)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("n", [3, 6, 17])
def test_standard_simplex(n, mode):
    # points e_1..e_n: r = sqrt((n-1)/n), c = centroid, all multipliers 1/n
    c, r, info = ripalm.meb_solve(np.eye(n), None, 1e-10, mode)
    assert abs(r - np.sqrt((n - 1) / n)) <= 1e-9
    np.testing.assert_allclose(c, np.full(n, 1.0 / n), atol=1e-8)
    if mode == "fp64":
        np.testing.assert_allclose(info["U"], np.full(n, 1.0 / n), atol=1e-6)


@pytest.mark.parametrize("mode", MODES)
def test_cross_polytope_and_interior_points(mode):
    # +-e_j lie on the unit sphere and their hull contains its centre: r = 1, c = 0
    d = 5
    rng = np.random.default_rng(3)
    inner = rng.standard_normal((200, d))
    inner *= (0.9 * rng.uniform(0, 1, 200) / np.sqrt((inner ** 2).sum(1)))[:, None]
    C = np.vstack([np.eye(d), -np.eye(d), inner]) * 3.0 + 7.0      # scaled and shifted
    c, r, _ = ripalm.meb_solve(C, None, 1e-10, mode)
    assert abs(r - 3.0) <= 1e-8
    np.testing.assert_allclose(c, np.full(d, 7.0), atol=1e-7)


@pytest.mark.parametrize("mode", MODES)
def test_degenerate_inputs(mode):
    # single ball
    c, r, _ = ripalm.meb_solve(np.array([[1.0, -2.0, 3.0]]), np.array([0.25]), 1e-10, mode)
    assert abs(r - 0.25) <= 1e-9 and np.allclose(c, [1, -2, 3], atol=1e-8)
    # all centres equal: r = max r_i
    C = np.tile(np.array([[0.5, 0.5]]), (9, 1)); R = np.linspace(0.1, 0.9, 9)
    c, r, _ = ripalm.meb_solve(C, R, 1e-10, mode)
    assert abs(r - 0.9) <= 1e-9 and np.allclose(c, [0.5, 0.5], atol=1e-8)
    # all balls are the same point: r = 0
    c, r, _ = ripalm.meb_solve(np.ones((4, 3)), None, 1e-10, mode)
    assert r == 0.0 and np.allclose(c, 1.0)
    # one ball contains all the others: that ball
    rng = np.random.default_rng(4)
    C = np.vstack([[0.3, -0.1, 0.2], rng.uniform(-1, 1, (30, 3))]); R = np.r_[10.0, rng.uniform(0, 1, 30)]
    c, r, _ = ripalm.meb_solve(C, R, 1e-10, mode)
    assert abs(r - 10.0) <= 1e-8 and np.allclose(c, C[0], atol=1e-7)
    # duplicated balls change nothing
    C = rng.standard_normal((20, 3)); R = rng.uniform(0, 0.5, 20)
    c1, r1, _ = ripalm.meb_solve(C, R, 1e-10, mode)
    c2, r2, _ = ripalm.meb_solve(np.vstack([C, C, C]), np.r_[R, R, R], 1e-10, mode)
    assert abs(r1 - r2) <= 1e-8 * r1 and np.allclose(c1, c2, atol=1e-7)


@pytest.mark.parametrize("mode", MODES)
def test_bruteforce_plane(mode):
    """Every 1-, 2- and 3-ball support subset in d = 2 (60 random instances, m <= 8)."""
    rng = np.random.default_rng(2024)
    worst = 0.0
    for trial in range(60):
        m = int(rng.integers(2, 9))
        C = rng.uniform(-1, 1, (m, 2)) * rng.choice([0.1, 1.0, 30.0])
        kind = trial % 4
        if kind == 0:
            R = None                                   # points
        elif kind == 1:
            R = rng.uniform(0, 0.5, m)
        elif kind == 2:
            R = rng.uniform(0, 0.5, m); C[1] = C[0]    # duplicate centre
        else:
            R = rng.uniform(0, 2.0, m)                 # big balls: containment happens
        bc, br = bruteforce_meb_2d(C, R)
        c, r, info = ripalm.meb_solve(C, R, 1e-10, mode)
        assert info["converged"], (trial, info["phases"][-1][2].history)
        worst = max(worst, abs(r - br) / br, np.linalg.norm(c - bc) / (1 + br))
        assert abs(r - br) <= 2e-9 * br, (trial, r, br)
        assert np.linalg.norm(c - bc) <= 2e-6 * (1 + br), (trial, c, bc)
    assert worst < 2e-6


def _check_certificate_and_invariants(C, R, c, r, info, tol):
    m, d = C.shape
    Rz = np.zeros(m) if R is None else R
    # containment (upper bound): r is the smallest feasible radius for c
    dist = np.sqrt(((C - c) ** 2).sum(1)) + Rz
    assert dist.max() <= r * (1 + 1e-15) and abs(dist.max() - r) <= 1e-15 * r
    U, V = info["U"], info["V"]
    I = info["index_set"]
    Cs, Rs = (C, Rz) if I is None else (C[I], Rz[I])
    # dual cone feasibility and the stationarity part of the KKT system
    assert np.all(U >= 0) and np.all(np.sqrt((V ** 2).sum(1)) <= U * (1 + 1e-12) + 1e-300)
    assert abs(U.sum() - 1) <= 10 * tol and np.linalg.norm(V.sum(0)) <= 10 * tol
    # weak duality: LB <= r* <= r   (a reduced problem is a relaxation: its LB is valid too)
    lb = dual_lower_bound(Cs, Rs, U, V)
    assert lb <= r * (1 + 1e-12)
    assert r - lb <= 50 * tol * (1 + r), (r, lb)
    # the centre is the multiplier-weighted mean of the touching points (KKT)
    sup = U > 1e-9
    assert 1 <= sup.sum() <= d + 1 + 5
    w = Cs[sup] - c
    p = Cs[sup] + Rs[sup][:, None] * w / np.sqrt((w ** 2).sum(1))[:, None]
    cc = (U[sup][:, None] * p).sum(0) / U[sup].sum()
    assert np.linalg.norm(cc - c) <= 1e-5 * (1 + r)
    return lb


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("k,m,d", [(1, 10_000, 10), (2, 20_000, 100), (3, 1_500, 1000), (5, 300, 2000)])
def test_certificate_on_config_distributions(k, m, d, mode):
    C, R = workloads.config(k, m, d)
    c, r, info = ripalm.meb_solve(C, R, 1e-8, mode)
    assert info["converged"]
    _check_certificate_and_invariants(C, R, c, r, info, 1e-8)
    if mode == "mixed":
        assert info["rounds"] == 1 and info["n_red"][0] < m
        c64, r64, _ = ripalm.meb_solve(C, R, 1e-10, "fp64")
        assert abs(r - r64) <= 1e-8 * r64


def test_config4_boundary_heavy():
    # half of the points on the unit sphere: r* = 1, c* = 0; the screen keeps the sphere half plus
    # the interior points with ||p|| >= 0.98:  0.5 + 0.5 (1 - (0.98/0.99)^32) = 0.6388 of m
    m, d = 40_000, 32
    C, R = workloads.config(4, m, d)
    c, r, info = ripalm.meb_solve(C, R, 1e-8, "mixed")
    assert abs(r - 1.0) <= 1e-8 and np.linalg.norm(c) <= 1e-6
    frac = info["n_red"][0] / m
    want = 0.5 + 0.5 * (1 - (0.98 / 0.99) ** 32)
    assert abs(frac - want) <= 0.01


def _table1():
    rows = {}
    with open(os.path.join(GOLDEN, "paper_table1_kept.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(s) for s in line.split()]
            rows[v[0]] = v[1:]
    return rows


def test_paper_table1_kept_counts():
    """P:L326-333.  Counting {i : s_i <= 0.02 r*} at the solution of the paper's instances
    reproduces Table 1 (pins screen_flags, tol_red = 0.02 r_hat [reading 9], the instance
    generator and the solver's radius).  The paper's own counts come from ITS approximate
    float32 ball, so a couple of entries may differ by a few balls: >= 17 of 20 must be exact
    and all within 3%."""
    table = _table1()
    ms = [1000, 5000, 10000, 50000, 100000]
    exact = 0
    for d, want in table.items():
        sol = {}
        for m, w in zip(ms, want):
            C, R = workloads.paper_instance(m, d)
            key = min(m, 4096)          # the generator has period 4096: m >= 4096 repeats the same balls
            if key not in sol:
                cs, rs, info = ripalm.meb_solve(C[:5000], R[:5000], 1e-10, "fp64")
                assert info["converged"]
                sol[key] = (cs, rs)
            cs, rs = sol[key]
            flags, _ = prim.screen_flags(C.astype(np.float32), R.astype(np.float32), rs, cs, 0.02 * rs)
            got = int(flags.sum())
            exact += int(got == w)
            assert abs(got - w) <= max(2, 0.03 * w), (d, m, got, w)
    assert exact >= 17, exact


def test_paper_instances_mixed_flow():
    """The full mixed flow on two of the paper's instances keeps about Table 1's number of balls,
    needs one refinement round, and agrees with the FP64 run."""
    table = _table1()
    for d, m, col in [(20, 1000, 0), (40, 5000, 1)]:
        C, R = workloads.paper_instance(m, d)
        c, r, info = ripalm.meb_solve(C, R, 1e-8, "mixed")
        c64, r64, _ = ripalm.meb_solve(C, R, 1e-10, "fp64")
        assert info["converged"] and info["rounds"] == 1
        assert abs(info["n_red"][0] - table[d][col]) <= 0.25 * table[d][col] + 3
        assert abs(r - r64) <= 1e-8 * r64


def test_accelerated_gradient_inner_solver_reaches_the_subproblem_minimiser():
    """a first-order inner solver minimises the same strongly convex Psi_k as Algorithm 2, so with the
    stopping tests tightened both must stop at the same point (the minimiser of (4) is unique)."""
    rng = np.random.default_rng(31)
    C = rng.standard_normal((400, 6)); R = rng.uniform(0, 0.2, 400)
    c0, L = ripalm.initial_point(C, R, ripalm.Params())
    Cn, Rn = (C - c0) / L, R / L
    x0 = np.zeros(7); x0[0] = 1.0
    U = np.zeros(400); V = np.zeros((400, 6))
    par = ripalm.Params(rho=0.0, ag_inner_max=20000)          # rho = 0: condition (5) never fires, only the KKT test does
    st1, st2 = ripalm.Stats(), ripalm.Stats()
    xa, eva, sa = ripalm.accelerated_gradient(Cn, Rn, U, V, x0, x0, x0, 4.0, 1.0, -1.0, par, np.float64, L, st1)
    xs, evs, ss = ripalm.ssn(Cn, Rn, U, V, x0, x0, x0, 4.0, 1.0, -1.0, par, np.float64, L, st2)
    assert np.linalg.norm(evs["grad"]) <= 1e-9                 # Newton reached the minimiser of Psi_k
    assert np.linalg.norm(eva["grad"]) <= 1e-6 and st1.evals > st2.evals
    assert np.linalg.norm(xa - xs) <= 1e-6 * (1 + np.linalg.norm(xs))
    assert abs(eva["psi_var"] - evs["psi_var"]) <= 1e-10 * abs(evs["psi_var"])


@pytest.mark.parametrize("mode", MODES)
def test_first_outer_iterations_by_accelerated_gradient_same_optimum(mode):
    """The inner solver is a path choice: with the first two outer iterations solved by the accelerated gradient
    method the unique optimum is the same (closed form: regular simplex, and brute force in the plane)."""
    par = ripalm.Params(ag_outer=2)
    n = 9
    c, r, info = ripalm.meb_solve(np.eye(n), None, 1e-10, mode, par)
    assert info["converged"] and abs(r - np.sqrt((n - 1) / n)) <= 1e-9
    rng = np.random.default_rng(32)
    C = rng.uniform(-1, 1, (7, 2)); R = rng.uniform(0, 0.4, 7)
    c, r, info = ripalm.meb_solve(C, R, 1e-10, mode, par)
    cb, rb = bruteforce_meb_2d(C, R)
    assert abs(r - rb) <= 1e-8 * rb and np.linalg.norm(c - cb) <= 1e-6
