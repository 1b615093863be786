"""GPU parity tests of the per-primitive entry points against the CPU oracle (run with -m gpu).

Bar (BASELINE.json north_star): FP64 reductions within 1e-12 and FP32
within 1e-5 of the oracle, relative to the sum of |terms| of the reduction; per-ball outputs within
the same tolerance of sigma-free magnitudes |a_i| + nb_i; integer work (compaction, argmax, index
sets given flags) bit-exact.  Counts and flags may differ only on balls within the tolerance of a
branch / threshold boundary; the tests evaluate at generic points and list those balls.

Balls near a branch boundary (SURVEY.md section 8(c) "Parity metrics": "balls within
10 tol_p of a branch or threshold boundary may land on the other side"): the evaluation point of
`make_state` is moved off the data by a factor 1.0001 and such balls are MASKED out of the per-ball,
count and list comparisons -- the two sides evaluate ||b_i|| with different summation orders, so which
side of `nb <= a` a ball within rounding of the boundary lands on is not defined by the paper.  The
REDUCTIONS get no allowance for them: Pi_Q is continuous, so a ball that flips branch changes its own
terms of psi, the gradient and the multiplier sums only in second order (t -> 0 at the B2/B3 boundary,
lam -> 1 at the B1/B3 boundary).  Only P_i (hvp, dense H) jumps across a boundary; there the allowance
is the listed balls' own bound sigma ||P_i||_F.
"""
import numpy as np
import pytest
import torch

from oracle import primitives as prim
from tests._gpu_common import dvec, make_state, to_device

pytestmark = pytest.mark.gpu

TOL = {0: 1e-12, 1: 1e-5}
NPDT = {0: np.float64, 1: np.float32}
THDT = {0: torch.float64, 1: torch.float32}

# (m, d, ld_pad): spans every row mapping of the streaming kernel (G x CPT tiles, the loop kernel,
# the unaligned scalar path), several tiles per warp and a ragged last tile
SHAPES = [(1000, 10, 0), (4999, 32, 0), (3001, 100, 0), (777, 1000, 0), (70, 2600, 0), (257, 33, 0),
          (64, 3, 1), (33, 1, 0), (1500, 20, 4), (513, 257, 1),
          # lane groups of the tile kernel's gradient part (2, 4, 8 or 16 lanes per row) and its 384-thread
          # instance (stages of 8 KB and more: 256-byte rows in FP64 and FP32, 1024-byte rows)
          (1203, 5, 0), (2000, 64, 0), (1031, 128, 0), (999, 16, 0)]


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


@pytest.fixture(scope="module")
def ctx(meb):
    c = meb.Context(1 << 17, 4096)
    yield c
    c.close()


def _near_boundary(ev, tol):
    a, nb = ev["a"].astype(np.float64), ev["nb"].astype(np.float64)
    scale = np.abs(a) + nb
    return (np.abs(nb - a) <= 10 * tol * scale) | (np.abs(nb + a) <= 10 * tol * scale)


def _branch_flip_slack(C, R, U, V, x, sigma, prec):
    """Allowance for balls within the tolerance of a branch boundary of P:L115, whose P_i may
    legitimately be taken from the other branch: sigma * ||P_i||_F <= sigma * sqrt(d+1) each."""
    ev = prim.eval_alm(C, R, U, V, x, x, sigma, 0.0, dtype=NPDT[prec])
    return float(_near_boundary(ev, TOL[prec]).sum()) * sigma * np.sqrt(C.shape[1] + 1.0)


def _check_eval(meb, ctx, prec, C, R, U, V, x, xbar, sigma, tau, layout, ld_pad):
    tol = TOL[prec]
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], layout, ld_pad)
    if layout == "none":
        U = np.zeros_like(U); V = np.zeros_like(V)
    res = meb.meb_eval_alm(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), sigma, tau,
                           per_ball=True, active=True)
    ev = prim.eval_alm(C, R, U, V, x, xbar, sigma, tau, dtype=NPDT[prec])
    s = res["scalars"].cpu().numpy()
    g = res["grad"].cpu().numpy()
    near = _near_boundary(ev, tol)
    E = meb.EV
    # per-ball outputs
    t_gpu, lam_gpu = res["t"].cpu().numpy(), res["lam"].cpu().numpy()
    mag = np.abs(ev["a"].astype(np.float64)) + ev["nb"].astype(np.float64) + 1e-300
    ok = ~near
    assert np.all(np.abs(t_gpu - ev["t"])[ok] <= tol * mag[ok])
    assert np.all(np.abs(lam_gpu - ev["lam"])[ok] <= 4 * tol)
    # branch counts and the active list: exact away from the boundaries
    act_o = np.flatnonzero(ev["br"] != 2)
    act_g = res["active_idx"].cpu().numpy()
    assert np.all(np.diff(act_g) > 0)
    diff = np.setxor1d(act_o, act_g)
    assert np.all(near[diff])
    if not near.any():
        assert int(s[E["N_B1"]]) == ev["n_b1"] and int(s[E["N_B3"]]) == ev["n_b3"]
        assert int(s[E["N_ACTIVE"]]) == act_o.size
        lam_list = res["active_lam"].cpu().numpy()
        assert np.all(np.abs(lam_list - ev["lam"][act_o]) <= 4 * tol)
    # reductions, relative to the sum of |terms|.  No allowance for the `near` balls: every summand is a
    # continuous function of (a_i, nb_i) across the branch boundaries (see the module docstring)
    assert near.sum() <= (2 if prec == 0 else 12), int(near.sum())
    slack = 0.0
    assert abs(s[E["SUM_PROJ2"]] - ev["sum_proj2"]) <= tol * ev["scale_proj2"] + slack
    assert abs(s[E["SUM_UPLUS"]] - ev["sum_uplus"]) <= tol * ev["scale_uplus"] + slack
    assert abs(s[E["SUM_DMULT2"]] - ev["sum_dmult2"]) <= 4 * tol * ev["scale_dmult2"] + slack
    psi_scale = abs(x[0]) + 0.5 * sigma * ev["scale_proj2"] + 0.5 * tau / sigma * float((x - xbar) @ (x - xbar))
    assert abs(s[E["PSI"]] - ev["psi_var"]) <= tol * psi_scale + slack
    gscale = np.concatenate([[1 + ev["scale_uplus"]], ev["scale_vplus"]]) + tau / sigma * np.abs(x - xbar)
    assert np.linalg.norm(g - ev["grad"]) <= tol * np.linalg.norm(gscale) + slack
    nsv = float(np.sqrt(np.sum(ev["sum_vplus"] ** 2)))
    assert abs(s[E["NORM_SUM_VPLUS"]] - nsv) <= tol * np.linalg.norm(ev["scale_vplus"]) + slack
    # maxima: each per-ball value is within tol of its magnitude
    big = float(np.max(mag)) * max(1.0, sigma) * (1 + float(np.max(mag)))
    assert abs(s[E["MAX_PFEAS"]] - ev["max_pfeas"]) <= 4 * tol * float(np.max(mag))
    assert abs(s[E["MAX_COMPL"]] - ev["max_compl"]) <= 8 * tol * big
    assert s[E["MAX_DFEAS"]] <= 8 * tol * big
    return ev, res


@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
@pytest.mark.parametrize("layout", ["none", "sparse", "dense"])
def test_eval_alm_fp64(meb, ctx, m, d, ld_pad, layout):
    C, R, U, V, x, xbar = make_state(100 + m + d, m, d, with_radii=(m % 2 == 1))
    _check_eval(meb, ctx, 0, C, R, U, V, x, xbar, 2.5, 0.7, layout, ld_pad)


@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
@pytest.mark.parametrize("layout", ["none", "sparse"])
def test_eval_alm_fp32(meb, ctx, m, d, ld_pad, layout):
    C, R, U, V, x, xbar = make_state(200 + m + d, m, d, with_radii=(m % 2 == 0))
    # the FP32 entry point takes float data: round the inputs once, both sides see the same floats
    C = C.astype(np.float32).astype(np.float64); U = U.astype(np.float32).astype(np.float64)
    V = V.astype(np.float32).astype(np.float64)
    R = None if R is None else R.astype(np.float32).astype(np.float64)
    _check_eval(meb, ctx, 1, C, R, U, V, x, xbar, 1.5, 1.0, layout, ld_pad)


def test_eval_alm_deterministic(meb, ctx):
    C, R, U, V, x, xbar = make_state(7, 20000, 48)
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, torch.float64, "sparse")
    outs = []
    for _ in range(3):
        r = meb.meb_eval_alm(ctx, 0, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), 2.0, 1.0)
        outs.append((r["scalars"].cpu().numpy().copy(), r["grad"].cpu().numpy().copy()))
    for s, g in outs[1:]:
        assert np.array_equal(s, outs[0][0]) and np.array_equal(g, outs[0][1])     # same bits


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("m,d,ld_pad", [(1000, 10, 0), (3001, 100, 0), (777, 1000, 0), (70, 2600, 0), (257, 33, 0)])
def test_hvp(meb, ctx, prec, m, d, ld_pad):
    C, R, U, V, x, xbar = make_state(300 + m + d, m, d)
    if prec == 1:
        C = C.astype(np.float32).astype(np.float64); U = U.astype(np.float32).astype(np.float64)
        V = V.astype(np.float32).astype(np.float64); R = R.astype(np.float32).astype(np.float64)
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], "sparse", ld_pad)
    q = np.random.default_rng(5).standard_normal(d + 1)
    Hq = meb.meb_hvp(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), 2.0, 0.5, dvec(q)).cpu().numpy()
    want, scale = prim.hvp(C, R, U, V, x, 2.0, 0.5, q, dtype=NPDT[prec])
    slack = _branch_flip_slack(C, R, U, V, x, 2.0, prec) * np.linalg.norm(q)
    assert np.linalg.norm(Hq - want) <= 4 * TOL[prec] * np.linalg.norm(scale) + slack
    assert q @ Hq >= 0.25 * (q @ q) * (1 - 1e-6)          # q^T H q >= (tau/sigma) ||q||^2


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("m,d", [(1000, 10), (4999, 32), (3001, 100), (600, 128), (257, 33),
                                 # syrk8_kernel (d <= 48): B = 2, 4, 6 with ragged column counts, many tiles per CTA
                                 (90_001, 16), (70_003, 27), (50_000, 48), (5, 3)])
def test_dense_hessian(meb, ctx, prec, m, d):
    C, R, U, V, x, xbar = make_state(400 + m + d, m, d)
    if prec == 1:
        C = C.astype(np.float32).astype(np.float64); U = U.astype(np.float32).astype(np.float64)
        V = V.astype(np.float32).astype(np.float64); R = R.astype(np.float32).astype(np.float64)
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], "sparse")
    H = meb.meb_dense_hessian(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), 2.0, 0.5).cpu().numpy()
    want, scale = prim.dense_hessian(C, R, U, V, x, 2.0, 0.5, dtype=NPDT[prec])
    slack = _branch_flip_slack(C, R, U, V, x, 2.0, prec)
    assert np.linalg.norm(H - want) <= 4 * TOL[prec] * np.linalg.norm(scale) + slack
    assert np.array_equal(H, H.T) or np.abs(H - H.T).max() <= 1e-13 * np.abs(H).max()


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("m,d", [(1000, 10), (3001, 100), (300, 1000), (40, 2600), (257, 33),
                                 # d <= 32: eight lanes per entry, four entries per warp and step (writev_short_kernel);
                                 # 120,001 balls are several sweeps of the grid and a ragged last step
                                 (4999, 32), (1203, 5), (999, 16), (120_001, 20), (3, 1)])
def test_update_multipliers(meb, ctx, prec, m, d):
    C, R, U, V, x, xbar = make_state(500 + m + d, m, d)
    if prec == 1:
        C = C.astype(np.float32).astype(np.float64); U = U.astype(np.float32).astype(np.float64)
        V = V.astype(np.float32).astype(np.float64); R = R.astype(np.float32).astype(np.float64)
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], "sparse")
    res = meb.meb_update_multipliers(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), 1.7)
    Up, Vp, m2 = prim.update_multipliers(C, R, U, V, x, 1.7, dtype=NPDT[prec])
    ev = prim.eval_alm(C, R, U, V, x, x, 1.7, 1.0, dtype=NPDT[prec])
    near = _near_boundary(ev, TOL[prec])          # balls that may legitimately land in the other branch
    ok = ~near
    Ug = res["U"].cpu().numpy().astype(np.float64)
    sl = res["v_slot"].cpu().numpy()
    Vg = res["Vrows"].cpu().numpy().astype(np.float64)
    mag = 1.7 * (np.abs(ev["a"].astype(np.float64)) + ev["nb"].astype(np.float64))
    assert np.all(np.abs(Ug - Up)[ok] <= TOL[prec] * mag[ok] + 1e-300)
    act = np.flatnonzero(ev["br"] != 2)
    act_g = np.flatnonzero(sl >= 0)
    assert np.all(near[np.setxor1d(act, act_g)])
    assert res["n_slots"] == act_g.size and res["code"] == 0
    assert np.array_equal(sl[act_g], np.arange(act_g.size))          # rows in ascending ball order
    both = np.intersect1d(act, act_g)
    both = both[ok[both]]
    assert np.all(np.abs(Vg[sl[both]] - Vp[both]) <= TOL[prec] * mag[both][:, None])
    assert np.all(Ug[sl < 0] == 0)
    assert abs(res["sum_mult2"] - m2) <= 4 * TOL[prec] * m2          # continuous across the branch boundaries
    act = act_g
    # capacity error: too few rows for the active balls
    res2 = meb.meb_update_multipliers(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), 1.7, cap_rows=act.size - 1)
    assert res2["code"] == meb.MEB_E_CAPACITY and res2["n_slots"] == act.size


@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
def test_feasibility_check(meb, ctx, m, d, ld_pad):
    C, R, U, V, x, xbar = make_state(600 + m + d, m, d, with_radii=(m % 2 == 1))
    Cd, Rd, *_ = to_device(C, R, U, V, torch.float64, "none", ld_pad)
    r, c = x[0], x[1:]
    eps = 0.05
    dmax, amax, viol_idx, viol = prim.feasibility_check(C, R, r, c, eps)
    res = meb.meb_feasibility_check(ctx, Cd, Rd, r, dvec(c), eps)
    scale = np.abs(viol + r).max() + abs(r)
    assert abs(res["delta_max"] - dmax) <= 1e-12 * scale
    top = np.flatnonzero(viol >= dmax - 1e-12 * scale)
    assert res["argmax"] in top
    near = np.abs(viol - eps) <= 1e-12 * scale
    got = res["viol_idx"].cpu().numpy()
    assert np.all(np.diff(got) > 0) and np.all(near[np.setxor1d(got, viol_idx)])
    # kept mask removes kept balls from the violated set (V subset of the discarded balls)
    kept = np.zeros(m, dtype=np.uint8); kept[viol_idx[::2]] = 1
    res2 = meb.meb_feasibility_check(ctx, Cd, Rd, r, dvec(c), eps, torch.from_numpy(kept).cuda())
    _, _, v2, _ = prim.feasibility_check(C, R, r, c, eps, kept)
    assert np.all(near[np.setxor1d(res2["viol_idx"].cpu().numpy(), v2)])
    # too small an output list
    if viol_idx.size > 1 and not near.any():
        res3 = meb.meb_feasibility_check(ctx, Cd, Rd, r, dvec(c), eps, cap=1)
        assert res3["code"] == meb.MEB_E_CAPACITY and res3["n_viol"] == viol_idx.size
        assert res3["viol_idx"].cpu().numpy()[0] == viol_idx[0]


def test_feasibility_argmax_tie_smallest_index(meb, ctx):
    C = np.zeros((300, 4)); C[17] = [2, 0, 0, 0]; C[250] = [0, 0, -2, 0]; C[99] = [0, 2, 0, 0]
    Cd = torch.from_numpy(C).cuda()
    res = meb.meb_feasibility_check(ctx, Cd, None, 1.0, dvec(np.zeros(4)), 0.5)
    assert res["delta_max"] == 1.0 and res["argmax"] == 17
    assert list(res["viol_idx"].cpu().numpy()) == [17, 99, 250]


@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
def test_screen_compact(meb, ctx, m, d, ld_pad):
    C, R, U, V, x, xbar = make_state(700 + m + d, m, d, with_radii=(m % 2 == 1))
    C32 = C.astype(np.float32); R32 = None if R is None else R.astype(np.float32)
    Cd, Rd, *_ = to_device(C32.astype(np.float64), None if R is None else R32.astype(np.float64), U, V,
                           torch.float32, "none", ld_pad)
    r_hat, c_hat = x[0], x[1:]
    # threshold chosen so that about 40% of the balls are retained whatever d is (distances concentrate)
    dist = np.sqrt(((C32.astype(np.float64) - c_hat) ** 2).sum(1)) + (0 if R is None else R32)
    tol_red = float(np.quantile(r_hat - dist, 0.4)) + 1e-4 * r_hat
    flags, s = prim.screen_flags(C32, R32, r_hat, c_hat, tol_red)
    res = meb.meb_screen_compact(ctx, Cd, Rd, r_hat, dvec(c_hat), tol_red)
    fg = res["flags"].cpu().numpy()
    near = np.abs(s.astype(np.float64) - tol_red) <= 1e-5 * (abs(r_hat) + np.abs(s) + 1)
    assert np.all(near[fg != flags])                               # flags agree away from the threshold
    # bit-exact compaction of the flags the GPU itself computed
    assert np.array_equal(res["idx"].cpu().numpy(), np.flatnonzero(fg).astype(np.int32))
    assert res["count"] == int(fg.sum()) and 0 < res["count"] < m


@pytest.mark.parametrize("m", [1, 31, 32, 33, 1000, 65536, 65537, 131072, 100003])
@pytest.mark.parametrize("density", [0.0, 0.01, 0.5, 1.0])
def test_compaction_bit_exact_given_flags(meb, ctx, m, density):
    rng = np.random.default_rng(m + int(100 * density))
    flags = (rng.uniform(size=m) < density).astype(np.uint8)
    fd = torch.from_numpy(flags).cuda()
    res = meb.meb_screen_compact(ctx, None, None, 0.0, None, 0.0, flags=fd, flags_are_input=True)
    want = prim.compact(flags)
    assert res["count"] == want.size
    assert np.array_equal(res["idx"].cpu().numpy(), want)
    if want.size > 3:                                              # capacity error keeps the prefix
        res2 = meb.meb_screen_compact(ctx, None, None, 0.0, None, 0.0, cap=3, flags=fd, flags_are_input=True)
        assert res2["code"] == meb.MEB_E_CAPACITY and res2["count"] == want.size
        assert np.array_equal(res2["idx"].cpu().numpy(), want[:3])


@pytest.mark.parametrize("m,d,ld_pad", SHAPES)
def test_ingest(meb, ctx, m, d, ld_pad):
    from oracle import ripalm
    C, R, U, V, x, xbar = make_state(800 + m + d, m, d, with_radii=(m % 2 == 1))
    Cd, Rd, *_ = to_device(C, R, U, V, torch.float64, "none", ld_pad)
    res = meb.meb_ingest(ctx, Cd, Rd, 1024, want_shadow=True)
    c0, L = ripalm.initial_point(C, R, ripalm.Params())
    assert np.abs(res["c0"].cpu().numpy() - c0).max() <= 1e-13 * (1 + np.abs(C).max())
    assert abs(res["L"] - L) <= 1e-12 * L and res["n_bad"] == 0
    sh = res["C32"].cpu().numpy()
    want = (C - res["c0"].cpu().numpy()[None, :]).astype(np.float32)
    assert np.array_equal(sh, want)                                # fl32(c_i - c0), element by element
    if R is not None:
        assert np.array_equal(res["R32"].cpu().numpy(), R.astype(np.float32))


def test_ingest_flags_bad_input(meb, ctx):
    C, R, *_ = make_state(9, 500, 12)
    C[123, 4] = np.nan
    R[400] = -0.1
    res = meb.meb_ingest(ctx, torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda())
    assert res["n_bad"] == 2


def test_argument_errors(meb, ctx):
    lib = meb.load()
    assert lib.meb_eval_alm(ctx.h, 0, 10, 3, None, 3, None, None, None, None, 0, None, None, 1.0, 1.0,
                            None, None, None, None, None, None, None) == meb.MEB_E_ARG
    C = torch.zeros((10, 3), dtype=torch.float64, device="cuda")
    x = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(meb.MebError):
        meb.meb_eval_alm(ctx, 0, C, None, None, None, None, x, x, -1.0, 1.0)       # sigma <= 0
    big = meb.Context(16, 4)
    with pytest.raises(meb.MebError) as ei:
        meb.meb_eval_alm(big, 0, torch.zeros((17, 3), dtype=torch.float64, device="cuda"), None, None, None,
                         None, x, x, 1.0, 1.0)
    assert ei.value.code == meb.MEB_E_CAPACITY
    big.close()


def test_compaction_multi_segment_path(meb):
    """Masks above 2M balls take the two-kernel segmented compaction (count + ranked write)."""
    m = 2_500_003
    rng = np.random.default_rng(77)
    flags = (rng.uniform(size=m) < 0.3).astype(np.uint8)
    flags[-1] = 1
    fd = torch.from_numpy(flags).cuda()
    with meb.Context(m, 4) as big:
        res = meb.meb_screen_compact(big, None, None, 0.0, None, 0.0, flags=fd, flags_are_input=True)
    want = prim.compact(flags)
    assert res["count"] == want.size and np.array_equal(res["idx"].cpu().numpy(), want)


def test_small_solver_and_graph_agree(meb):
    """The single-CTA solver (m <= 4096) and the graph path (MEB_NO_SMALL=1) reach the same optimum."""
    import os
    import workloads
    C, R = workloads.config(1, 3000, 10)
    dC, dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
    with meb.Context(3000, 10) as c1:
        ca, ra, sta = meb.meb_solve(c1, dC, dR, 1e-8, meb.MEB_MODE_FP64)
    os.environ["MEB_NO_SMALL"] = "1"
    try:
        with meb.Context(3000, 10) as c2:
            cb, rb, stb = meb.meb_solve(c2, dC, dR, 1e-8, meb.MEB_MODE_FP64)
    finally:
        del os.environ["MEB_NO_SMALL"]
    assert sta["converged"] == 1 and stb["converged"] == 1
    assert abs(ra - rb) <= 1e-9 * rb and np.linalg.norm(ca.numpy() - cb.numpy()) <= 1e-6 * (1 + rb)
    assert sta["kernel_launches"] < stb["kernel_launches"]


@pytest.mark.parametrize("prec", [0, 1])
def test_eval_alm_unaligned_scalar_arrays(meb, ctx, prec):
    """R, U and the slot map start at addresses that are not multiples of 16 bytes: the tile kernel must
    then read them from global memory instead of staging them with bulk copies (same results)."""
    m, d = 3001, 100
    C, R, U, V, x, xbar = make_state(911, m, d)
    if prec == 1:
        C = C.astype(np.float32).astype(np.float64); U = U.astype(np.float32).astype(np.float64)
        V = V.astype(np.float32).astype(np.float64); R = R.astype(np.float32).astype(np.float64)
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], "sparse")
    ref = meb.meb_eval_alm(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), 2.0, 0.5, per_ball=True)

    def shifted(t):
        buf = torch.empty(t.numel() + 1, dtype=t.dtype, device=t.device)
        buf[1:].copy_(t)
        return buf[1:]
    Rs, Us, Ss = shifted(Rd), shifted(Ud), shifted(slot)
    assert Rs.data_ptr() % 16 != 0 and Ss.data_ptr() % 16 != 0
    got = meb.meb_eval_alm(ctx, prec, Cd, Rs, Us, Ss, Vr, dvec(x), dvec(xbar), 2.0, 0.5, per_ball=True)
    assert torch.equal(ref["scalars"], got["scalars"]) and torch.equal(ref["grad"], got["grad"])
    assert torch.equal(ref["t"], got["t"]) and torch.equal(ref["lam"], got["lam"])


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("m,d,ld_pad", [(1000, 10, 0), (4999, 32, 0), (3001, 100, 0), (1031, 128, 0), (777, 1000, 0),
                                        (70, 2600, 0), (1500, 20, 4)])
@pytest.mark.parametrize("layout", ["none", "sparse"])
def test_eval_alm_multi(meb, ctx, prec, m, d, ld_pad, layout):
    """Multi-trial evaluation: psi at x and at x - gamma_k Delta from ONE pass, against the
    oracle's plain loop of evaluations.  The expansion ||b + g dc||^2 = ||b||^2 + 2 g <b, dc> + g^2 ||dc||^2 loses
    a few ulps to cancellation, hence 8 tol_p."""
    C, R, U, V, x, xbar = make_state(900 + m + d, m, d, with_radii=(m % 2 == 1))
    if prec == 1:
        f = lambda a: None if a is None else a.astype(np.float32).astype(np.float64)
        C, R, U, V = f(C), f(R), f(U), f(V)
    rng = np.random.default_rng(m + d)
    direction = np.concatenate([[-0.08 * x[0]], 0.05 * rng.standard_normal(d) / np.sqrt(d)])
    gammas = [0.5, 0.75, 0.875, 0.9375]
    Cd, Rd, Ud, slot, Vr = to_device(C, R, U, V, THDT[prec], layout, ld_pad)
    if layout == "none":
        U = np.zeros_like(U); V = np.zeros_like(V)
    if (Cd.stride(0) * Cd.element_size()) % 16 != 0:
        # rows that are not 16-byte aligned go to the scalar-load kernels, which carry no multi-trial code
        with pytest.raises(meb.MebError) as ei:
            meb.meb_eval_alm_multi(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), 2.5, 0.7, dvec(direction), gammas)
        assert ei.value.code == meb.MEB_E_CAPACITY
        return
    res = meb.meb_eval_alm_multi(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), 2.5, 0.7, dvec(direction), gammas)
    ref = meb.meb_eval_alm(ctx, prec, Cd, Rd, Ud, slot, Vr, dvec(x), dvec(xbar), 2.5, 0.7)
    assert torch.equal(res["scalars"][:12], ref["scalars"][:12]) and torch.equal(res["grad"], ref["grad"])
    want = prim.eval_alm_line(C, R, U, V, x, xbar, 2.5, 0.7, direction, gammas, dtype=NPDT[prec])
    got = res["psi"].cpu().numpy()
    for k, (psi, scale) in enumerate(want):
        assert abs(got[k] - psi) <= 8 * TOL[prec] * scale, (k, got[k], psi, scale)
    # the points differ: the predictions are not all the same number
    assert len({float(v) for v in got}) == len(gammas)
