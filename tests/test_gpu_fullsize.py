"""Parity at BASELINE.json's full size, in the launch configuration bench.py times (config 2:
m = 1e6 points in R^100, mixed precision; run with -m gpu).

* whole solve: the returned ball is feasible to 1e-10 (1 + r) (checked on the host over all m), and its
  radius is within 1e-8 of the optimum by a two-sided argument that needs no full-size oracle run:
  MEB(subset) <= MEB(all) <= r_gpu for ANY subset, and the oracle (run to 1e-10) on the balls within
  2% of the returned boundary gives MEB(subset); r_gpu <= (1 + 1e-8) MEB(subset) closes the sandwich.
* eval_alm (FP32, the dominant kernel of the bench): per-ball outputs of sampled balls against the
  oracle evaluated one ball at a time, and the reductions against the oracle's full pass.
"""
import numpy as np
import pytest
import torch

import workloads
from oracle import primitives as prim
from oracle import ripalm

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def meb():
    import paper_2605_31425_b200 as meb
    meb.load()
    return meb


@pytest.fixture(scope="module")
def config2():
    C, R = workloads.config(2)                      # 1e6 x 100, points
    return C, torch.from_numpy(C).cuda()


def test_full_size_mixed_solve_sandwich(meb, config2):
    C, dC = config2
    m, d = C.shape
    with meb.Context(m, d) as ctx:
        c, r, st = meb.meb_solve(ctx, dC, None, 1e-8, meb.MEB_MODE_MIXED)
    c = c.numpy()
    assert st["converged"] == 1 and st["passes_fp32_full"] > 0 and st["rounds"] >= 1
    dist = np.sqrt(((C - c[None, :]) ** 2).sum(axis=1))
    assert dist.max() - r <= 1e-10 * (1 + r)                       # feasible for ALL m balls
    near = np.flatnonzero(dist >= 0.98 * r)                        # a subset that contains the support
    assert 0 < near.size < 5000
    cs, rs, info = ripalm.meb_solve(C[near], None, 1e-10, "fp64")
    assert info["converged"]
    assert rs <= r * (1 + 1e-12)                                   # MEB(subset) <= MEB(all) <= r
    assert r - rs <= 1e-8 * rs                                     # ... and r is within 1e-8 of it
    assert np.linalg.norm(c - cs) <= 1e-5 * (1 + rs)


def test_full_size_eval_fp32_sampled_and_reduced(meb, config2):
    C, dC = config2
    m, d = C.shape
    rng = np.random.default_rng(3)
    with meb.Context(m, d) as ctx:
        ing = meb.meb_ingest(ctx, dC, None, 1024, want_shadow=True)
        C32 = ing["C32"]
        L = ing["L"]
        x = np.concatenate([[0.93 * L], 0.01 * rng.standard_normal(d)])     # generic point, ~2% of the balls active
        xd = torch.from_numpy(x).cuda()
        sigma, tau = 1.0 / L, 1.0 / L ** 2
        res = meb.meb_eval_alm(ctx, meb.MEB_FP32, C32, None, None, None, None, xd, xd, sigma, tau, per_ball=True)
        s = res["scalars"].cpu().numpy()
        g = res["grad"].cpu().numpy()
        t_gpu = res["t"].cpu().numpy()
        lam_gpu = res["lam"].cpu().numpy()
    Ch = C32.cpu().numpy().astype(np.float64)                      # the very floats the kernel read
    zero = np.zeros(m)
    ev = prim.eval_alm(Ch, None, zero, np.zeros((m, d), dtype=np.float32), x, x, sigma, tau, dtype=np.float32)
    a, nb = ev["a"].astype(np.float64), ev["nb"].astype(np.float64)
    mag = np.abs(a) + nb
    near = (np.abs(nb - a) <= 1e-4 * mag) | (np.abs(nb + a) <= 1e-4 * mag)
    # sampled balls, one by one
    for i in rng.choice(m, 2000, replace=False):
        if near[i]:
            continue
        one = prim.eval_alm(Ch[i:i + 1], None, zero[:1], np.zeros((1, d), dtype=np.float32), x, x, sigma, tau,
                            dtype=np.float32)
        assert abs(t_gpu[i] - float(one["t"][0])) <= 1e-5 * mag[i]
        assert abs(lam_gpu[i] - float(one["lam"][0])) <= 4e-5
    # reductions of the whole pass, relative to the sums of |terms|
    E = meb.EV
    slack = 0.0            # the summands are continuous across the branch boundaries (tests/test_gpu_primitives.py)
    assert abs(s[E["SUM_PROJ2"]] - ev["sum_proj2"]) <= 1e-5 * ev["scale_proj2"] + slack
    assert abs(s[E["SUM_UPLUS"]] - ev["sum_uplus"]) <= 1e-5 * ev["scale_uplus"] + slack
    gscale = np.concatenate([[1 + ev["scale_uplus"]], ev["scale_vplus"]])
    assert np.linalg.norm(g - ev["grad"]) <= 1e-5 * np.linalg.norm(gscale) + slack
    if not near.any():
        assert int(s[E["N_B3"]]) == ev["n_b3"] and int(s[E["N_B1"]]) == ev["n_b1"]


# ------------------------------------------------------------------------------------------------
# Configs 3, 4, 5 at BASELINE.json's full size ("What's missing" 4).  These sizes reach
# paths the small parity cases do not: long-row kernels over 0.8-16 GB (byte offsets above 2^31), the
# two-kernel segmented compaction inside a solve (config 4 keeps 6.4e6 balls), V pools of 5e6 rows and
# their growth (ST_NEED_CAPACITY relaunch), the reduced solve at d = 1e3 / 1e4.
# ------------------------------------------------------------------------------------------------
def _generate(k):
    m, d, has_r = workloads.CONFIG_SHAPES[k]
    C = np.empty((m, d), dtype=np.float64)
    R = np.empty(m, dtype=np.float64) if has_r else None
    workloads.config_into(k, C, R, m, d, 0, threads=8)
    return C, R


def _upload(C, R):
    """Row blocks through a bounded staging tensor (a 16 GB torch.from_numpy(...).cuda() would pin nothing and
    still works, but block copies keep the host footprint at the instance itself)."""
    m, d = C.shape
    dC = torch.empty((m, d), dtype=torch.float64, device="cuda")
    step = max(1, (256 << 20) // (8 * d))
    for r0 in range(0, m, step):
        dC[r0:r0 + step].copy_(torch.from_numpy(C[r0:r0 + step]))
    dR = None if R is None else torch.from_numpy(R).cuda()
    return dC, dR


def _dist_plus_radius(C, R, c):
    """||c_i - c|| + r_i for every ball, block by block (plain numpy on the host)."""
    m, d = C.shape
    out = np.empty(m)
    step = max(1, (512 << 20) // (8 * d))
    for r0 in range(0, m, step):
        blk = C[r0:r0 + step] - c[None, :]
        out[r0:r0 + step] = np.sqrt(np.einsum("ij,ij->i", blk, blk))
    if R is not None:
        out += R
    return out


def _sandwich(meb, C, R, modes, near_max):
    """Feasibility of the returned ball over ALL m balls, and its radius within 1e-8 of the optimum by
    MEB(subset) <= MEB(all) <= r_gpu with the oracle (run to 1e-10) on the balls within 2% of the boundary."""
    m, d = C.shape
    dC, dR = _upload(C, R)
    out = {}
    with meb.Context(m, d) as ctx:
        for mode in modes:
            pm = meb.MEB_MODE_MIXED if mode == "mixed" else meb.MEB_MODE_FP64
            c, r, st = meb.meb_solve(ctx, dC, dR, 1e-8, pm)
            out[mode] = (c.numpy().copy(), r, st)
    del dC, dR
    torch.cuda.empty_cache()
    sub = None
    for mode, (c, r, st) in out.items():
        assert st["converged"] == 1, (mode, st["kkt"])
        reach = _dist_plus_radius(C, R, c)
        assert reach.max() - r <= 1e-10 * (1 + r), (mode, reach.max() - r)      # feasible for ALL m balls
        if sub is None:                                                          # one oracle run serves both modes
            near = np.flatnonzero(reach >= 0.98 * r)
            assert 0 < near.size <= near_max, near.size
            cs, rs, info = ripalm.meb_solve(C[near], None if R is None else R[near], 1e-10, "fp64",
                                            ripalm.Params(dense_d_max=1024))      # dense Newton up to d = 1000: a path choice
            assert info["converged"]
            sub = (cs, rs)
        cs, rs = sub
        assert rs <= r * (1 + 1e-12), (mode, r, rs)                              # MEB(subset) <= MEB(all) <= r
        assert r - rs <= 1e-8 * rs, (mode, r, rs)
        assert np.linalg.norm(c - cs) <= 1e-5 * (1 + rs)
    return out


def test_full_size_config3_sandwich(meb):
    C, R = _generate(3)                               # 1e5 balls in R^1000: matrix-free Newton path
    out = _sandwich(meb, C, R, ["mixed", "fp64"], near_max=8000)
    st = out["mixed"][2]
    assert st["passes_fp32_full"] > 0 and st["rounds"] >= 1 and 0 < st["n_reduced"] < 20000
    assert out["fp64"][2]["cg_iters"] > 0 or out["fp64"][2]["newton_iters"] > 0


def test_full_size_config5_sandwich(meb):
    C, R = _generate(5)                               # 2e5 balls in R^10000: 16 GB of centres
    out = _sandwich(meb, C, R, ["mixed", "fp64"], near_max=200)
    st = out["mixed"][2]
    assert st["passes_fp32_full"] > 0 and st["rounds"] >= 1 and 0 < st["n_reduced"] <= 200
    assert st["pass_bytes"][meb.PASS["INGEST"]] >= 16e9 * 1.4         # 16 GB read + 8 GB shadow written


def test_full_size_config4_closed_form(meb):
    """Config 4: half of the 1e7 points lie on the unit sphere (their hull contains the origin), the rest inside
    the 0.99-ball, so r* = 1 and c* = 0 up to the rounding of the generated unit vectors,
    and the retain rule at 0.02 r keeps 0.5 + 0.5 (1 - (0.98/0.99)^32) = 0.6388 of the balls."""
    C, R = _generate(4)
    m, d = C.shape
    dC, _ = _upload(C, None)
    with meb.Context(m, d) as ctx:
        for mode, pm in (("fp64", meb.MEB_MODE_FP64), ("mixed", meb.MEB_MODE_MIXED)):
            c, r, st = meb.meb_solve(ctx, dC, None, 1e-8, pm)
            c = c.numpy()
            assert st["converged"] == 1, (mode, st["kkt"])
            assert abs(r - 1.0) <= 1e-8 and np.linalg.norm(c) <= 1e-6, (mode, r, np.linalg.norm(c))
            reach = _dist_plus_radius(C, None, c)
            assert reach.max() - r <= 1e-10 * (1 + r)
            if mode == "mixed":
                want = 0.5 + 0.5 * (1.0 - (0.98 / 0.99) ** 32)
                assert abs(st["n_reduced"] / m - want) <= 0.002, st["n_reduced"] / m
                assert st["n_reduced"] > 2_100_000                     # the segmented (multi-kernel) compaction ran
            else:
                assert st["n_support"] >= 4_000_000                    # V pools grew from 4096 rows to millions


def test_full_size_config4_eval_with_multiplier_rows(meb):
    """FP64 eval_alm at config 4's size with a multiplier row for each of the 5e6 sphere points (the slowest
    streaming path: pool rows are read next to the centre rows): reductions against the oracle's full pass,
    per-ball outputs of sampled balls against the oracle evaluated one ball at a time."""
    C, _ = _generate(4)
    m, d = C.shape
    rng = np.random.default_rng(5)
    nrm = np.sqrt(np.einsum("ij,ij->i", C, C))
    on = np.flatnonzero(nrm > 0.995)                                   # the sphere points, ascending
    assert abs(on.size - m // 2) == 0
    U = np.zeros(m)
    U[on] = rng.uniform(0.5, 1.5, on.size) / on.size
    Vrows = C[on] * (U[on] * rng.uniform(0.2, 1.0, on.size))[:, None]  # ||v_i|| <= u_i
    slot = np.full(m, -1, dtype=np.int32)
    slot[on] = np.arange(on.size, dtype=np.int32)                      # ascending ball order, as the update writes them
    x = np.concatenate([[1.0005], 1e-3 * rng.standard_normal(d)])
    xbar = x + 1e-3 * rng.standard_normal(d + 1)
    sigma, tau = 50.0, 1.0
    dC, _ = _upload(C, None)
    with meb.Context(m, d) as ctx:
        res = meb.meb_eval_alm(ctx, meb.MEB_FP64, dC, None, torch.from_numpy(U).cuda(), torch.from_numpy(slot).cuda(),
                               torch.from_numpy(Vrows).cuda(), torch.from_numpy(x).cuda(), torch.from_numpy(xbar).cuda(),
                               sigma, tau, per_ball=True)
        s = res["scalars"].cpu().numpy(); g = res["grad"].cpu().numpy()
        t_gpu = res["t"].cpu().numpy(); lam_gpu = res["lam"].cpu().numpy()
    del dC
    torch.cuda.empty_cache()
    V = np.zeros((m, d))
    V[on] = Vrows
    ev = prim.eval_alm(C, None, U, V, x, xbar, sigma, tau)
    a, nb = ev["a"], ev["nb"]
    mag = np.abs(a) + nb
    near = (np.abs(nb - a) <= 1e-11 * mag) | (np.abs(nb + a) <= 1e-11 * mag)
    assert near.sum() <= 2
    E = meb.EV
    assert ev["n_b3"] > 500_000
    assert abs(s[E["SUM_PROJ2"]] - ev["sum_proj2"]) <= 1e-12 * ev["scale_proj2"]
    assert abs(s[E["SUM_UPLUS"]] - ev["sum_uplus"]) <= 1e-12 * ev["scale_uplus"]
    assert abs(s[E["SUM_DMULT2"]] - ev["sum_dmult2"]) <= 4e-12 * ev["scale_dmult2"]
    gscale = np.concatenate([[1 + ev["scale_uplus"]], ev["scale_vplus"]]) + tau / sigma * np.abs(x - xbar)
    assert np.linalg.norm(g - ev["grad"]) <= 1e-12 * np.linalg.norm(gscale)
    if not near.any():
        assert int(s[E["N_B3"]]) == ev["n_b3"] and int(s[E["N_B1"]]) == ev["n_b1"]
    for i in rng.choice(m, 3000, replace=False):
        if near[i]:
            continue
        one = prim.eval_alm(C[i:i + 1], None, U[i:i + 1], V[i:i + 1], x, xbar, sigma, tau)
        assert abs(t_gpu[i] - float(one["t"][0])) <= 1e-12 * mag[i]
        assert abs(lam_gpu[i] - float(one["lam"][0])) <= 4e-12
