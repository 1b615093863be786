"""Pins for oracle/primitives.py (CPU only): each reduction is checked against something that
is not the oracle's own formula -- a ball-by-ball Python loop written from the paper's
definitions, central finite differences, or an inequality the paper states."""
import math

import numpy as np
import pytest

import workloads
from oracle import primitives as prim
from oracle import soc


def _state(rng, m, d, with_radii=True, frac_mult=0.3):
    """A generic (non-converged) evaluation point with multipliers inside Q."""
    C = rng.standard_normal((m, d))
    R = rng.uniform(0, 0.3, m) if with_radii else None
    c = rng.standard_normal(d) * 0.1
    dist = np.sqrt(((C - c) ** 2).sum(1)) + (0 if R is None else R)
    r = float(np.quantile(dist, 0.7))            # 30% of the balls stick out
    x = np.concatenate([[r], c])
    xbar = x + rng.standard_normal(d + 1) * 0.05
    U = np.zeros(m)
    V = np.zeros((m, d))
    k = int(frac_mult * m)
    idx = rng.permutation(m)[:k]
    U[idx] = rng.uniform(0.01, 1.0, k)
    dirs = rng.standard_normal((k, d))
    dirs /= np.sqrt((dirs ** 2).sum(1))[:, None]
    V[idx] = dirs * (U[idx] * rng.uniform(0, 1, k))[:, None]    # ||v_i|| <= u_i
    return C, R, U, V, x, xbar


def _loop_eval(C, R, U, V, x, xbar, sigma, tau):
    """Ball-by-ball evaluation straight from P:L107, L111, L115, L139, L309 (pure Python)."""
    m, d = C.shape
    r, c = x[0], x[1:]
    psi_sum = 0.0
    su = 0.0
    sv = np.zeros(d)
    dm = 0.0
    n1 = n3 = 0
    mp = mc = 0.0
    for i in range(m):
        ri = 0.0 if R is None else R[i]
        a = ri - r + U[i] / sigma
        b = C[i] - c + V[i] / sigma
        nb = math.sqrt(float(b @ b))
        if nb <= a:
            p0, p1 = a, b.copy(); n1 += 1
        elif nb <= -a:
            p0, p1 = 0.0, np.zeros(d)
        else:
            s = (a + nb) / 2
            p0, p1 = s, s * b / nb; n3 += 1
        psi_sum += p0 * p0 + float(p1 @ p1)
        up, vp = sigma * p0, sigma * p1
        su += up
        sv += vp
        dm += (up - U[i]) ** 2 + float((vp - V[i]) @ (vp - V[i]))
        # primal cone distance of (r - r_i, c - c_i)
        a2, b2 = r - ri, c - C[i]
        n2 = math.sqrt(float(b2 @ b2))
        if n2 <= a2:
            dist = 0.0
        elif n2 <= -a2:
            dist = math.sqrt(a2 * a2 + n2 * n2)
        else:
            dist = (n2 - a2) / math.sqrt(2)
        mp = max(mp, dist)
        mc = max(mc, abs(a2 * up + float(b2 @ vp)))
    dx = x - xbar
    psi = r + sigma / 2 * psi_sum + tau / (2 * sigma) * float(dx @ dx)
    g = np.concatenate([[1 - su], -sv]) + tau / sigma * dx
    return psi, g, dm, n1, n3, mp, mc


@pytest.mark.parametrize("with_radii", [True, False])
def test_eval_alm_against_loop(with_radii):
    rng = np.random.default_rng(11)
    C, R, U, V, x, xbar = _state(rng, 300, 5, with_radii)
    sigma, tau = 2.5, 0.7
    ev = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau)
    psi, g, dm, n1, n3, mp, mc = _loop_eval(C, R, U, V, x, xbar, sigma, tau)
    assert n3 > 20 and ev["n_b3"] == n3 and ev["n_b1"] == n1
    assert abs(ev["psi_var"] - psi) <= 1e-12 * abs(psi)
    np.testing.assert_allclose(ev["grad"], g, atol=1e-12 * (1 + np.abs(g).max()))
    assert abs(ev["sum_dmult2"] - dm) <= 1e-12 * dm
    assert abs(ev["max_pfeas"] - mp) <= 1e-14 and abs(ev["max_compl"] - mc) <= 1e-13
    assert ev["max_dfeas"] <= 1e-15 * (1 + np.abs(ev["Uplus"]).max())   # sigma*Pi(z) lies in Q


def test_eval_alm_has_b1_balls():
    # a ball whose shifted point lies inside Q needs a big multiplier: u/sigma > ||b|| + r - r_i
    rng = np.random.default_rng(12)
    C, R, U, V, x, xbar = _state(rng, 50, 3)
    U[:5] = 50.0
    ev = prim.eval_alm(C, R, U, V, x, xbar, 1.0, 1.0)
    psi, g, dm, n1, n3, mp, mc = _loop_eval(C, R, U, V, x, xbar, 1.0, 1.0)
    assert n1 >= 5 and ev["n_b1"] == n1
    np.testing.assert_allclose(ev["grad"], g, rtol=1e-12, atol=1e-12)


def test_gradient_is_derivative_of_psi():
    """grad = d psi / dx, by central differences (psi is C^1, piecewise C^2)."""
    rng = np.random.default_rng(13)
    C, R, U, V, x, xbar = _state(rng, 400, 6)
    sigma, tau = 3.0, 1.3
    ev = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau)
    h = 1e-6
    fd = np.empty_like(x)
    for j in range(x.size):
        e = np.zeros_like(x); e[j] = h
        fp = prim.eval_alm(C, R, U, V, x + e, xbar, sigma, tau)["psi_var"]
        fm = prim.eval_alm(C, R, U, V, x - e, xbar, sigma, tau)["psi_var"]
        fd[j] = (fp - fm) / (2 * h)
    np.testing.assert_allclose(ev["grad"], fd, atol=2e-6 * (1 + np.abs(fd).max()))


def test_hvp_is_derivative_of_gradient_and_matches_dense():
    rng = np.random.default_rng(14)
    C, R, U, V, x, xbar = _state(rng, 120, 4)
    sigma, tau = 2.0, 0.5
    a, B, *_ = prim.shifted_points(C, R, U, V, x, sigma)
    nb = soc.row_norms(B)
    assert np.min(np.abs(nb - np.abs(a))) > 1e-4          # generic point: off the kinks
    H, _ = prim.dense_hessian(C, R, U, V, x, sigma, tau)
    Hloop = prim.dense_hessian_loop(C, R, U, V, x, sigma, tau)
    np.testing.assert_allclose(H, Hloop, atol=1e-12 * np.abs(Hloop).max())
    np.testing.assert_allclose(H, H.T, atol=1e-13)
    h = 1e-6
    for j in range(x.size):
        e = np.zeros_like(x); e[j] = 1.0
        Hq, _ = prim.hvp(C, R, U, V, x, sigma, tau, e)
        np.testing.assert_allclose(Hq, Hloop[:, j], atol=1e-12 * np.abs(Hloop).max())
        gp = prim.eval_alm(C, R, U, V, x + h * e, xbar, sigma, tau)["grad"]
        gm = prim.eval_alm(C, R, U, V, x - h * e, xbar, sigma, tau)["grad"]
        np.testing.assert_allclose((gp - gm) / (2 * h), Hq, atol=5e-6 * np.abs(Hloop).max())
    # SPD with smallest eigenvalue >= tau/sigma
    assert np.linalg.eigvalsh(H).min() >= tau / sigma * (1 - 1e-12)
    q = rng.standard_normal(x.size)
    Hq, _ = prim.hvp(C, R, U, V, x, sigma, tau, q)
    assert q @ Hq >= tau / sigma * (q @ q)


def test_update_multipliers_definition():
    rng = np.random.default_rng(15)
    C, R, U, V, x, xbar = _state(rng, 200, 4)
    sigma = 1.7
    Up, Vp, m2 = prim.update_multipliers(C, R, U, V, x, sigma)
    for i in range(0, 200, 7):
        a = R[i] - x[0] + U[i] / sigma
        b = C[i] - x[1:] + V[i] / sigma
        t, PV, _, _ = soc.proj_soc(np.array([a]), b[None, :])
        assert abs(Up[i] - sigma * t[0]) <= 1e-15 * (1 + abs(Up[i]))
        np.testing.assert_allclose(Vp[i], sigma * PV[0], atol=1e-15)
    assert np.all(Up >= 0) and np.all(np.sqrt((Vp ** 2).sum(1)) <= Up * (1 + 1e-14) + 1e-300)
    assert abs(m2 - float((Up ** 2).sum() + (Vp ** 2).sum())) <= 1e-12 * m2
    # u_i = 0  =>  v_i = 0 exactly: the fact the sparse V layout of the CUDA path rests on
    assert np.all(Vp[Up == 0] == 0)


def test_feasibility_check_definition():
    rng = np.random.default_rng(16)
    C = rng.standard_normal((500, 3)); R = rng.uniform(0, 0.2, 500)
    c = np.array([0.1, -0.2, 0.05]); r = 2.0
    dmax, amax, viol_idx, viol = prim.feasibility_check(C, R, r, c, 0.05)
    want = np.array([R[i] + math.dist(c, C[i]) - r for i in range(500)])
    np.testing.assert_allclose(viol, want, atol=1e-15)
    assert amax == int(np.argmax(want)) and dmax == want[amax]
    assert list(viol_idx) == [i for i in range(500) if want[i] > 0.05] and len(viol_idx) > 3
    kept = np.zeros(500, bool); kept[viol_idx[::2]] = True
    _, _, v2, _ = prim.feasibility_check(C, R, r, c, 0.05, kept)
    assert list(v2) == list(viol_idx[1::2])
    # ties: the smallest index wins
    C2 = np.array([[1.0, 0], [0, 1.0], [-1.0, 0]]); d2, a2, _, _ = prim.feasibility_check(C2, None, 0.5, np.zeros(2), 0)
    assert a2 == 0 and d2 == 0.5


def test_screen_and_compact():
    rng = np.random.default_rng(17)
    C = rng.standard_normal((1000, 8)).astype(np.float32); R = rng.uniform(0, 0.1, 1000).astype(np.float32)
    c_hat = np.zeros(8); r_hat = 4.0
    flags, s = prim.screen_flags(C, R, r_hat, c_hat, 0.5)
    s64 = r_hat - R.astype(np.float64) - np.sqrt((C.astype(np.float64) ** 2).sum(1))
    np.testing.assert_allclose(s, s64, atol=2e-6)                # float32 slack
    far = np.abs(s64 - 0.5) > 1e-5
    assert np.array_equal(flags[far].astype(bool), (s64 <= 0.5)[far]) and 5 < flags.sum() < 995
    idx = prim.compact(flags)
    assert idx.dtype == np.int32 and list(idx) == [i for i in range(1000) if flags[i]]


def test_fp32_mode_close_to_fp64():
    rng = np.random.default_rng(18)
    C, R, U, V, x, xbar = _state(rng, 2000, 16)
    e64 = prim.eval_alm(C, R, U, V, x, xbar, 2.0, 1.0)
    e32 = prim.eval_alm(C, R, U, V, x, xbar, 2.0, 1.0, dtype=np.float32)
    assert e32["Uplus"].dtype == np.float32
    assert abs(e32["psi_var"] - e64["psi_var"]) <= 1e-5 * abs(e64["psi_var"])
    assert np.linalg.norm(e32["sum_vplus"] - e64["sum_vplus"]) <= 1e-5 * np.linalg.norm(e64["scale_vplus"])


def test_paper_instance_generator():
    """psi_0 = 7, psi_{j+1} = (445 psi_j + 1) mod 4096, values psi_j/40.96 from j = 1,
    order r_1, c_1(1..d), r_2, ..."""
    C, R = workloads.paper_instance(3, 2)
    psi = [7]
    for _ in range(9):
        psi.append((445 * psi[-1] + 1) % 4096)
    # by hand: 445*7+1 = 3116;  445*3116+1 = 1386621 = 338*4096 + 2173;  445*2173+1 = 966986 = 236*4096 + 330
    assert psi[1:4] == [3116, 2173, 330]
    seq = [p / 40.96 for p in psi[1:]]
    assert R[0] == seq[0] and list(C[0]) == seq[1:3] and R[1] == seq[3] and list(C[2]) == seq[7:9]
    Cb, Rb = workloads.paper_instance(5000, 20)
    assert 0 <= Cb.min() and Cb.max() < 100 and Rb.max() < 100


def _state32(seed, m, d):
    """A state whose data are exactly representable in float32 (both modes see the same numbers)."""
    rng = np.random.default_rng(seed)
    C, R, U, V, x, xbar = _state(rng, m, d)
    f = lambda a: a.astype(np.float32).astype(np.float64)
    return f(C), f(R), f(U), f(V), x, xbar


def test_fp32_mode_of_hvp_close_to_fp64():
    """The low-precision mode (DESIGN reading 8: float32 data and per-ball arithmetic, float64 sums) of hvp
    against its float64 mode on the same float32-representable data: within 1e-5 of the sum of |terms|.
    A wrong cast in the q1 / rho path moves the result by far more."""
    C, R, U, V, x, _ = _state32(21, 1500, 12)
    q = np.random.default_rng(22).standard_normal(13)
    H64, scale = prim.hvp(C, R, U, V, x, 2.0, 0.5, q)
    H32, scale32 = prim.hvp(C, R, U, V, x, 2.0, 0.5, q, dtype=np.float32)
    assert H32.dtype == np.float64 and np.linalg.norm(scale) > 10
    assert np.linalg.norm(H32 - H64) <= 1e-5 * np.linalg.norm(scale)
    assert np.linalg.norm(H32 - H64) > 0                          # it did run in float32
    assert np.linalg.norm(scale32 - scale) <= 1e-5 * np.linalg.norm(scale)
    # unit vectors pick single columns of H: every entry of the FP32-mode operator is pinned
    Hd, sd = prim.dense_hessian(C, R, U, V, x, 2.0, 0.5)
    for j in (0, 1, 12):
        e = np.zeros(13); e[j] = 1.0
        col, _ = prim.hvp(C, R, U, V, x, 2.0, 0.5, e, dtype=np.float32)
        assert np.linalg.norm(col - Hd[:, j]) <= 1e-5 * np.linalg.norm(sd[:, j])


def test_fp32_mode_of_dense_hessian_close_to_fp64():
    C, R, U, V, x, _ = _state32(23, 1200, 9)
    H64, scale = prim.dense_hessian(C, R, U, V, x, 1.5, 0.8)
    H32, _ = prim.dense_hessian(C, R, U, V, x, 1.5, 0.8, dtype=np.float32)
    assert np.linalg.norm(H32 - H64) <= 1e-5 * np.linalg.norm(scale)
    assert np.linalg.norm(H32 - H64) > 0
    np.testing.assert_allclose(H32, H32.T, atol=1e-12 * np.abs(H32).max())
    assert np.linalg.eigvalsh(H32).min() >= 0.8 / 1.5 * (1 - 1e-4)      # P:L193 survives the low precision


def test_fp32_mode_of_update_multipliers_close_to_fp64():
    C, R, U, V, x, _ = _state32(24, 1000, 7)
    sigma = 1.7
    U64, V64, m64 = prim.update_multipliers(C, R, U, V, x, sigma)
    U32, V32, m32 = prim.update_multipliers(C, R, U, V, x, sigma, dtype=np.float32)
    assert U32.dtype == np.float32 and V32.dtype == np.float32
    a, B, *_ = prim.shifted_points(C, R, U, V, x, sigma)
    mag = sigma * (np.abs(a) + soc.row_norms(B))
    far = np.abs(soc.row_norms(B) - np.abs(a)) > 1e-4 * (np.abs(a) + soc.row_norms(B))   # off the branch boundaries
    assert far.sum() > 900
    assert np.all(np.abs(U32 - U64)[far] <= 1e-5 * mag[far])
    assert np.all(np.abs(V32 - V64)[far] <= 1e-5 * mag[far][:, None])
    assert abs(m32 - m64) <= 1e-5 * m64 + (~far).sum() * float(mag.max()) ** 2
    assert np.all(V32[U32 == 0] == 0)


def test_initial_point_hand_example():
    """DESIGN reading 3: c0 = mean of the S = min(m, sample_rows) rows floor(k m / S), L = max_i(||c_i - c0|| + r_i).
    m = 5, S = 2 -> rows 0 and 2.  By hand: c0 = ((0,0) + (4,0))/2 = (2,0); ||c_i - c0|| + r_i =
    2+1, 8+0.5, 2+0, 3+2, sqrt(10)+0  ->  L = 8.5 (ball 1)."""
    from oracle import ripalm
    C = np.array([[0.0, 0.0], [10.0, 0.0], [4.0, 0.0], [2.0, 3.0], [-1.0, -1.0]])
    R = np.array([1.0, 0.5, 0.0, 2.0, 0.0])
    c0, L = ripalm.initial_point(C, R, ripalm.Params(sample_rows=2))
    assert np.array_equal(c0, [2.0, 0.0]) and L == 8.5
    # S = 3: rows floor(0), floor(5/3) = 1, floor(10/3) = 3 -> c0 = (12/3, 3/3) = (4, 1)
    c0, L = ripalm.initial_point(C, None, ripalm.Params(sample_rows=3))
    assert np.allclose(c0, [4.0, 1.0], atol=1e-15)
    assert abs(L - np.sqrt(37.0)) <= 1e-15 * 7                      # farthest point: (10,0) -> sqrt(36 + 1)
    # fewer balls than sample_rows: the mean of all of them
    c0, L = ripalm.initial_point(C, R, ripalm.Params())
    assert np.allclose(c0, C.mean(axis=0), atol=1e-15)
