"""GPU parity of meb_solve against the CPU oracle (run with -m gpu).

Bar: final radius within 1e-8 relative of the oracle run to 1e-10; feasibility violation of the
returned ball <= 1e-10 (1 + r); centre within 1e-5 (1 + r) (the centre is less well conditioned than
the radius).  Iteration paths, multipliers and index sets may differ (DESIGN reading 14): only the
unique optimum is compared, the rest is checked for validity."""
import numpy as np
import pytest
import torch

import workloads
from oracle import ripalm

pytestmark = pytest.mark.gpu

MODES = ["fp64", "mixed"]


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


def _solve(meb, C, R, mode, tol=1e-8, host=False):
    m, d = C.shape
    with meb.Context(m, d) as ctx:
        pm = meb.MEB_MODE_FP64 if mode == "fp64" else meb.MEB_MODE_MIXED
        if host:
            hc = torch.from_numpy(C).pin_memory()
            hr = None if R is None else torch.from_numpy(R).pin_memory()
            c, r, st = meb.meb_solve_host(ctx, hc, hr, tol, pm)
        else:
            dC = torch.from_numpy(C).cuda()
            dR = None if R is None else torch.from_numpy(R).cuda()
            c, r, st = meb.meb_solve(ctx, dC, dR, tol, pm)
    return c.numpy(), r, st


def _violation(C, R, c, r):
    Rz = 0 if R is None else R
    return float(np.max(np.sqrt(((C - c) ** 2).sum(1)) + Rz - r))


def _check_against_oracle(meb, C, R, mode, host=False):
    c, r, st = _solve(meb, C, R, mode, host=host)
    # the oracle solves its Newton systems densely here (a path choice, DESIGN reading 5; CG at d = 1000 takes minutes)
    co, ro, _ = ripalm.meb_solve(C, R, 1e-10, "fp64", ripalm.Params(dense_d_max=4096))
    assert st["converged"] == 1
    assert abs(r - ro) <= 1e-8 * ro, (r, ro)
    assert np.linalg.norm(c - co) <= 1e-5 * (1 + ro)
    assert _violation(C, R, c, r) <= 1e-10 * (1 + r)
    assert st["kkt"] <= 1e-8
    return c, r, st


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("k,m,d", [(1, 10_000, 10), (2, 30_000, 100), (3, 3_000, 1000), (4, 60_000, 32),
                                   (5, 400, 3000), (1, 777, 7), (3, 999, 129)])
def test_solve_matches_oracle(meb, k, m, d, mode):
    C, R = workloads.config(k, m, d)
    c, r, st = _check_against_oracle(meb, C, R, mode)
    if mode == "mixed":
        assert st["rounds"] >= 1 and 0 < st["n_reduced"] <= m
        assert st["passes_fp32_full"] > 0 and st["passes_reduced"] > 0


@pytest.mark.parametrize("mode", MODES)
def test_solve_host_entry_point(meb, mode):
    C, R = workloads.config(1, 5000, 10)
    _check_against_oracle(meb, C, R, mode, host=True)


@pytest.mark.parametrize("mode", MODES)
def test_paper_instances(meb, mode):
    for m, d in [(1000, 20), (5000, 40)]:
        C, R = workloads.paper_instance(m, d)
        _check_against_oracle(meb, C, R, mode)


@pytest.mark.parametrize("mode", MODES)
def test_closed_forms(meb, mode):
    # two balls (P: north_star): r = (||c1-c2|| + r1 + r2)/2, centre on the segment
    c1, r1 = np.array([1.0, 2.0, -1.0, 0.5]), 0.7
    c2, r2 = np.array([-2.0, 0.0, 3.0, 1.5]), 1.9
    dist = np.linalg.norm(c1 - c2)
    rw = (dist + r1 + r2) / 2
    cw = c1 + (rw - r1) * (c2 - c1) / dist
    c, r, _ = _solve(meb, np.array([c1, c2]), np.array([r1, r2]), mode, 1e-10)
    assert abs(r - rw) <= 1e-9 * rw and np.allclose(c, cw, atol=1e-7)
    # regular simplex e_1..e_n
    n = 12
    c, r, _ = _solve(meb, np.eye(n), None, mode, 1e-10)
    assert abs(r - np.sqrt((n - 1) / n)) <= 1e-9 and np.allclose(c, 1.0 / n, atol=1e-7)
    # points on a sphere whose hull contains the centre
    d = 6
    C = np.vstack([np.eye(d), -np.eye(d)]) * 2.5 - 1.0
    c, r, _ = _solve(meb, C, None, mode, 1e-10)
    assert abs(r - 2.5) <= 1e-8 and np.allclose(c, -1.0, atol=1e-6)


@pytest.mark.parametrize("mode", MODES)
def test_degenerate_inputs(meb, mode):
    c, r, _ = _solve(meb, np.array([[1.0, -2.0, 3.0]]), np.array([0.25]), mode)        # m = 1
    assert abs(r - 0.25) <= 1e-9 and np.allclose(c, [1, -2, 3], atol=1e-7)
    C = np.tile(np.array([[0.5, 0.5]]), (9, 1)); R = np.linspace(0.1, 0.9, 9)           # equal centres
    c, r, _ = _solve(meb, C, R, mode)
    assert abs(r - 0.9) <= 1e-8 and np.allclose(c, 0.5, atol=1e-7)
    c, r, _ = _solve(meb, np.ones((4, 3)), None, mode)                                 # L = 0
    assert r == 0.0 and np.allclose(c, 1.0)
    rng = np.random.default_rng(4)                                                     # containment
    C = np.vstack([[0.3, -0.1, 0.2], rng.uniform(-1, 1, (30, 3))]); R = np.r_[10.0, rng.uniform(0, 1, 30)]
    c, r, _ = _solve(meb, C, R, mode)
    assert abs(r - 10.0) <= 1e-7 and np.allclose(c, C[0], atol=1e-6)


def test_bad_input_is_reported(meb):
    C, R = workloads.config(1, 300, 10)
    C[5, 5] = np.inf
    with pytest.raises(meb.MebError) as ei:
        _solve(meb, C, R, "fp64")
    assert ei.value.code == meb.MEB_E_INPUT
    C, R = workloads.config(1, 300, 10)
    R[7] = -1.0
    with pytest.raises(meb.MebError) as ei:
        _solve(meb, C, R, "mixed")
    assert ei.value.code == meb.MEB_E_INPUT


def test_solve_is_deterministic(meb):
    C, R = workloads.config(1, 20_000, 10)
    a = _solve(meb, C, R, "mixed")
    b = _solve(meb, C, R, "mixed")
    assert a[1] == b[1] and np.array_equal(a[0], b[0])


def _solve_with(meb, C, R, mode, params=None, tol=1e-8):
    m, d = C.shape
    with meb.Context(m, d) as ctx:
        pm = meb.MEB_MODE_FP64 if mode == "fp64" else meb.MEB_MODE_MIXED
        dC = torch.from_numpy(C).cuda()
        dR = None if R is None else torch.from_numpy(R).cuda()
        c, r, st = meb.meb_solve(ctx, dC, dR, tol, pm, params=params)
    return c.numpy(), r, st


@pytest.mark.parametrize("k,m,d", [(2, 200_000, 100), (3, 20_000, 1000), (1, 50_000, 10)])
def test_cut_trials_do_not_change_the_result(meb, k, m, d, monkeypatch):
    """Armijo trials whose partial sum of Psi already exceeds Psi(x) are stopped early:
    they are rejections either way, so the iterates -- and the result, bit for bit -- are those of a
    run with the early stop switched off.  The first Newton step from the feasible start (no active
    ball, H = (tau/sigma) I) always produces such trials."""
    C, R = workloads.config(k, m, d)
    c1, r1, s1 = _solve_with(meb, C, R, "fp64")
    monkeypatch.setenv("MEB_NO_ABORT", "1")
    c0, r0, s0 = _solve_with(meb, C, R, "fp64")
    assert s1["passes_cut"] > 0 and s0["passes_cut"] == 0
    assert r1 == r0 and np.array_equal(c1, c0)
    # same iterates, hence the same Newton steps; the number of PASSES may differ: a trial that runs to the end
    # predicts the next halvings exactly, a cut one only bounds them, so it can skip fewer of them (reading 19)
    assert s1["newton_iters"] == s0["newton_iters"] and s1["outer_iters"] == s0["outer_iters"]
    assert s0["trials_skipped"] >= s1["trials_skipped"]


@pytest.mark.parametrize("mode", MODES)
def test_inner_loop_does_not_spin_at_the_rounding_floor(meb, mode):
    """Reading 6: once the Newton decrement is below what Psi can resolve the inner loop leaves; before,
    condition (5) could keep it running to its cap with line searches on rounding noise (hundreds of
    passes on the config 2 distribution)."""
    C, R = workloads.config(2, 60_000, 100)
    c, r, st = _check_against_oracle(meb, C, R, mode)
    assert st["passes_fp64_full"] + st["passes_fp32_full"] <= 90, st


def test_armijo_shrink_min_is_only_a_path_choice(meb):
    """armijo_shrink_min < 1/2 skips Armijo trials that the parabola through Psi(x), Psi'(x; Delta) and
    the failed trial predicts to fail; the iteration path changes, the optimum does not."""
    C, R = workloads.config(2, 50_000, 100)
    p = meb.meb_default_params()
    p.armijo_shrink_min = 0.125
    c1, r1, s1 = _solve_with(meb, C, R, "fp64", params=p)
    c0, r0, s0 = _solve_with(meb, C, R, "fp64")
    assert s1["converged"] == 1 and s0["converged"] == 1
    assert abs(r1 - r0) <= 1e-8 * r0 and np.linalg.norm(c1 - c0) <= 1e-5 * (1 + r0)


@pytest.mark.parametrize("factor,k,m,d", [(-0.3, 2, 40_000, 100), (-100.0, 1, 10_000, 10), (-0.05, 3, 4_000, 1000)])
def test_refinement_rounds_reintroduce_violated_balls(meb, factor, k, m, d):
    """violated discarded balls are added back without limit and the reduced problem is solved
    again.  A useless retain rule (a NEGATIVE tol_red factor keeps only balls far outside the coarse ball;
    -100 keeps none, in which case the farthest ball alone starts the reduced problem, as in the oracle)
    forces rounds >= 2, the growth of the reduced buffers beyond their first capacity and the re-introduction
    code; the answer is still the unique optimum."""
    C, R = workloads.config(k, m, d)
    p = meb.meb_default_params()
    p.tol_red_factor = factor
    c, r, st = _solve_with(meb, C, R, "mixed", params=p)
    co, ro, _ = ripalm.meb_solve(C, R, 1e-10, "fp64", ripalm.Params(dense_d_max=4096))
    assert st["converged"] == 1 and st["rounds"] >= 2, st
    assert abs(r - ro) <= 1e-8 * ro and np.linalg.norm(c - co) <= 1e-5 * (1 + ro)
    assert _violation(C, R, c, r) <= 1e-10 * (1 + r)
    assert st["n_reduced"] > 1024 or factor == -100.0 or m < 2048


def test_refinement_round_cap_reports_not_converged(meb):
    C, R = workloads.config(2, 20_000, 100)
    p = meb.meb_default_params()
    p.tol_red_factor = -0.3
    p.max_rounds = 1
    with meb.Context(*C.shape) as ctx:
        c, r, st = meb.meb_solve(ctx, torch.from_numpy(C).cuda(), None, 1e-8, meb.MEB_MODE_MIXED, params=p,
                                 allow_not_converged=True)
    assert st["converged"] == 0 and st["rounds"] == 1
    assert _violation(C, R, c.numpy(), r) <= 1e-10 * (1 + r)       # the returned radius is still the feasible one


def test_stepped_solve_equals_graph_solve_and_fills_event_times(meb):
    """MEB_OPT_STEPPED sequences the same kernels from the host: same bits, and every streaming launch is
    bracketed by a CUDA-event pair (meb_stats.pass_ev_*), which is what bench.py's roofline reads."""
    C, R = workloads.config(3, 5_000, 1000)
    dC, dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
    with meb.Context(*C.shape) as ctx:
        c0, r0, s0 = meb.meb_solve(ctx, dC, dR, 1e-8, meb.MEB_MODE_MIXED)
        meb.meb_set_option(ctx, meb.OPT["STEPPED"], True)
        c1, r1, s1 = meb.meb_solve(ctx, dC, dR, 1e-8, meb.MEB_MODE_MIXED)
        meb.meb_set_option(ctx, meb.OPT["STEPPED"], False)
    assert r0 == r1 and torch.equal(c0, c1)
    P = meb.PASS
    assert s0["pass_ev_count"][P["EVAL_FP32"]] == 0 and s0["pass_ev_count"][P["INGEST"]] == 1
    n32 = s1["pass_ev_count"][P["EVAL_FP32"]]
    assert n32 == s1["passes_fp32_full"] - 1 - s1["passes_cut"] or n32 > 0      # screen pass is its own class
    assert s1["pass_ev_ms"][P["EVAL_FP32"]] > 0 and s1["pass_ev_bytes"][P["EVAL_FP32"]] >= n32 * C.size * 4


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("k,m,d", [(1, 6_000, 10), (2, 20_000, 100), (3, 2_000, 1000)])
def test_accelerated_gradient_first_outer_iterations(meb, k, m, d, mode):
    """the first outer iterations may solve subproblem (4) with the accelerated gradient
    method instead of semismooth Newton (meb_params.ag_outer).  Only the path changes: same unique optimum."""
    C, R = workloads.config(k, m, d)
    p = meb.meb_default_params()
    p.ag_outer = 2
    c, r, st = _solve_with(meb, C, R, mode, params=p)
    co, ro, _ = ripalm.meb_solve(C, R, 1e-10, "fp64", ripalm.Params(dense_d_max=4096))
    assert st["converged"] == 1 and st["ag_iters"] > 0, st
    assert abs(r - ro) <= 1e-8 * ro and np.linalg.norm(c - co) <= 1e-5 * (1 + ro)
    assert _violation(C, R, c, r) <= 1e-10 * (1 + r)


@pytest.mark.parametrize("m,d,with_radii", [(1, 127, True), (5, 1000, True), (40, 300, False), (200, 517, True), (256, 130, False)])
def test_cluster_solver_matches_graph_path_and_oracle(meb, m, d, with_radii):
    """Few balls with long rows (m <= 256, d > 126) run in ONE thread-block cluster (csrc/meb_wide.cu); MEB_OPT_NO_SMALL
    sends the same instance through the graph of grid kernels.  Same optimum, far fewer launches; oracle parity as usual."""
    rng = np.random.default_rng(5000 + m + d)
    C = rng.standard_normal((m, d)) * np.linspace(0.2, 2.0, d)
    R = rng.lognormal(-2.0, 1.0, size=m) if with_radii else None
    dC = torch.from_numpy(C).cuda()
    dR = None if R is None else torch.from_numpy(R).cuda()
    with meb.Context(m, d) as c1:
        ca, ra, sta = meb.meb_solve(c1, dC, dR, 1e-8, meb.MEB_MODE_FP64)
        ca2, ra2, sta2 = meb.meb_solve(c1, dC, dR, 1e-8, meb.MEB_MODE_FP64)
    with meb.Context(m, d) as c2:
        meb.meb_set_option(c2, meb.OPT["NO_SMALL"], True)
        cb, rb, stb = meb.meb_solve(c2, dC, dR, 1e-8, meb.MEB_MODE_FP64)
    assert sta["converged"] == 1 and stb["converged"] == 1
    assert ra == ra2 and torch.equal(ca, ca2)                          # deterministic
    assert abs(ra - rb) <= 1e-9 * (1 + rb) and np.linalg.norm(ca.numpy() - cb.numpy()) <= 1e-6 * (1 + rb)
    if m > 1:
        assert sta["kernel_launches"] < stb["kernel_launches"]
    co, ro, _ = ripalm.meb_solve(C, R, 1e-10, "fp64", ripalm.Params(dense_d_max=4096))
    assert abs(ra - ro) <= 1e-8 * (1 + ro)
    assert np.linalg.norm(ca.numpy() - co) <= 1e-5 * (1 + ro)
    assert _violation(C, R, ca.numpy(), ra) <= 1e-10 * (1 + ra)


@pytest.mark.parametrize("k,m,d", [(3, 20_000, 1000), (5, 3_000, 4000)])
def test_fused_screening_keeps_the_same_balls(meb, k, m, d):
    """Long rows: the retain rule of the screening is applied by the LAST evaluation pass of the low-precision
    run instead of a pass of its own.  Same arithmetic on the same point: the kept set, and with it every later iterate,
    is bit-identical; one FP32 pass fewer."""
    C, R = workloads.config(k, m, d)[:2]
    dC, dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
    out = []
    for off in (False, True):
        with meb.Context(m, d) as ctx:
            meb.meb_set_option(ctx, meb.OPT["NO_FUSED_SCREEN"], off)
            out.append(meb.meb_solve(ctx, dC, dR, 1e-8, meb.MEB_MODE_MIXED))
    (ca, ra, sa), (cb, rb, sb) = out
    assert sa["converged"] == 1 and sb["converged"] == 1
    assert sa["n_reduced"] == sb["n_reduced"] and ra == rb and torch.equal(ca, cb)
    assert sa["passes_fp32_full"] == sb["passes_fp32_full"] - 1
    assert sa["pass_count"][meb.PASS["SCREEN"]] == 0 and sb["pass_count"][meb.PASS["SCREEN"]] == 1
